// mm_passB4.cuh — pass B for LONG y lines: one thread-block CLUSTER of Q CTAs per (TC columns, zpos).
//
// The y transform of Eq. 8's convolution on a zero-padded line of n = py points, of which only the
// first n/2 are non-zero.  One radix-Q decimation-in-frequency step splits it into Q INDEPENDENT transforms of
// length m = n/Q — block q holds the frequencies ky = Q k' + q:
//     x_q[i] = ( sum_{t < Q/2} a[i + t m] w_Q^(q t) ) w_n^(q i),      X[Q k' + q] = FFT_m(x_q)[k'],
// so CTA q of the cluster loads the whole input line of its columns (every CTA reads all n/2 rows: the re-reads hit
// L2, the CTAs of a cluster run at the same time), transforms, multiplies by K^ and transforms back entirely inside its
// own shared memory, on a tile of m rows — 1/Q of the full-line tile, so rows stay 32 bytes wide where a single CTA would
// be down to one 8-byte column (fp32, ny = 4096) or would not fit at all (fp64, ny = 4096).  The inverse of the
// radix-Q step needs all Q blocks:
//     out[i + t m] = sum_q z_q[i] w_Q^(-q t),   z_q[i] = IFFT_m(block q)[i] conj(w_n^(q i)),   t < Q/2 (cropped),
// and is done through DISTRIBUTED SHARED MEMORY: after a cluster barrier CTA q reads rows [q m/Q, (q+1) m/Q) of all Q
// tiles (its own and Q-1 remote ones) and stores the finished rows to S, in place.
//
// Tile element (row p, component c, column col) at s[c*m*TC + p*TC + col] (component-major: consecutive rows are
// contiguous, so the lanes of a stage — consecutive butterflies — touch consecutive 16- / 32-byte row segments:
// conflict-free); rows hold bit-reversed positions after the forward stages: row p of block q is frequency
// ky = Q*brev_m(p) + q.  The multiply stage reads its 8-row blocks cyclically rotated by the block index (DFT_8 ->
// real per-frequency multiply -> IDFT_8 commutes with a cyclic shift of the 8 rows; neighbouring blocks are 8*TC
// elements = a multiple of 128 bytes apart and would otherwise hit the same banks).  K^ is read in its
// symmetric-packed form (Kh).
// Everything is __host__ __device__: tests/host_emul runs the Q compute phases of a cluster one after the other and
// then the Q combine phases.
#pragma once
#include "mm_fft.cuh"
#include "mm_kernels.cuh"
#include "mm_kernels2.cuh"

namespace mm {

// w_n^k for any 0 <= k < n (the table holds k <= n/2)
template <typename T> MM_HD cx<T> tw_any(twiddles<T> tw, int k, int n)
{
    if (k <= n / 2) return tw.get(k, n);
    const cx<T> w = tw.get(k - n / 2, n);
    return mk<T>(-w.x, -w.y);
}

// (-i)^e a  (forward radix-4 weights w_4^e)
template <typename E> MM_HD E rot_m(E a, int e)
{
    e &= 3;
    if (e == 0) return a;
    if (e == 1) return mul_mi(a);
    if (e == 2) return a - a - a;
    return mul_pi(a);
}

// first stage of block q: load + radix-Q combine + twiddle w_n^(q row) + radix R over the m rows
template <typename T, int V, int R, int Q>
MM_HD void yB4_first(const Geom& g, const cx<T>* Sz, cx<T>* s, twiddles<T> tw, int q, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = TC;
    const int n = g.py, m = n / Q, sub = m / R, CS = m * TC;
    for (int f = tid; f < sub * LC; f += nthr) {
        const int lc = f & (LC - 1), i = f >> logLC;
        cx<T> pw[R], wq[R];
        if (R > 1 && i != 0) twiddle_powers<T, R>(tw.get(i, m), pw);
#pragma unroll
        for (int r = 0; r < R; r++) wq[r] = tw_any<T>(tw, (int)(((long)q * (i + r * sub)) & (n - 1)), n);
#pragma unroll 1
        for (int c = 0; c < 3; c++) {
            const cx<T>* src = Sz + (long)c * g.comp + (long)i * g.Lx + lc * V;
            cx<T>* dst = s + c * CS + i * pitch + lc * V;
            E a[R];
#pragma unroll
            for (int r = 0; r < R; r++) {
                a[r] = ldv<E, T>(src + (long)r * sub * g.Lx);
                if (Q == 4) a[r] = a[r] + rot_m<E>(ldv<E, T>(src + ((long)r * sub + m) * g.Lx), q);
                if (q != 0) a[r] = cmul(a[r], wq[r]);
            }
            rad<E, R>::fwd(a);
            if (R > 1 && i != 0) {
#pragma unroll
                for (int r = 1; r < R; r++) a[r] = cmul(a[r], pw[r]);
            }
#pragma unroll
            for (int r = 0; r < R; r++) stv<E, T>(dst + r * sub * pitch, a[r]);
        }
    }
}

// last stage of block q: inverse radix R, then z = y conj(w_n^(q row)), left in the tile for the cluster combine
template <typename T, int V, int R, int Q>
MM_HD void yB4_last(const Geom& g, cx<T>* s, twiddles<T> tw, int q, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = TC;
    const int n = g.py, m = n / Q, sub = m / R, CS = m * TC;
    for (int f = tid; f < sub * LC; f += nthr) {
        const int lc = f & (LC - 1), i = f >> logLC;
        cx<T> pw[R], wq[R];
        if (R > 1 && i != 0) twiddle_powers<T, R>(tw.get(i, m), pw);
#pragma unroll
        for (int r = 0; r < R; r++) wq[r] = tw_any<T>(tw, (int)(((long)q * (i + r * sub)) & (n - 1)), n);
#pragma unroll 1
        for (int c = 0; c < 3; c++) {
            cx<T>* p = s + c * CS + i * pitch + lc * V;
            E a[R];
#pragma unroll
            for (int r = 0; r < R; r++) a[r] = ldv<E, T>(p + r * sub * pitch);
            if (R > 1 && i != 0) {
#pragma unroll
                for (int r = 1; r < R; r++) a[r] = cmulc(a[r], pw[r]);
            }
            rad<E, R>::inv(a);
#pragma unroll
            for (int r = 0; r < R; r++) stv<E, T>(p + r * sub * pitch, q != 0 ? cmulc(a[r], wq[r]) : a[r]);
        }
    }
}

// middle radix-8 stage over the m rows of the tile (DIR 0 forward DIF, 1 inverse DIT)
template <typename T, int V, int DIR>
MM_HD void yB4_mid8(const Geom& g, cx<T>* s, int m, int Lc, twiddles<T> tw, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = TC, CS = m * TC;
    const int sub = Lc >> 3, logsub = ilog2(sub);
    for (int f = tid; f < (m >> 3) * LC; f += nthr) {
        const int lc = f & (LC - 1), b = f >> logLC;
        const int blk = b >> logsub, i = b & (sub - 1);
        cx<T> pw[8];
        if (i != 0) twiddle_powers<T, 8>(tw.get(i, Lc), pw);
        cx<T>* base = s + (blk * Lc + i) * pitch + lc * V;
#pragma unroll 1
        for (int c = 0; c < 3; c++) {
            cx<T>* p = base + c * CS;
            E v[8];
#pragma unroll
            for (int r = 0; r < 8; r++) v[r] = ldv<E, T>(p + r * sub * pitch);
            if (DIR == 0) {
                rad<E, 8>::fwd(v);
                if (i != 0) {
#pragma unroll
                    for (int r = 1; r < 8; r++) v[r] = cmul(v[r], pw[r]);
                }
            } else {
                if (i != 0) {
#pragma unroll
                    for (int r = 1; r < 8; r++) v[r] = cmulc(v[r], pw[r]);
                }
                rad<E, 8>::inv(v);
            }
#pragma unroll
            for (int r = 0; r < 8; r++) stv<E, T>(p + r * sub * pitch, v[r]);
        }
    }
}

// last forward radix-8 stage (Lc = 8) + multiply by K^ + first inverse stage; three components of one column in
// registers.  Row p of block q is ky = Q*brev_m(p) + q.
template <typename T, bool IS3D, int Q>
MM_HD void yB4_mul8(const Geom& g, cx<T>* s, const T* Kz, T sz, int q, int tid, int nthr)
{
    const int TC = g.TC, logTC = ilog2(TC), pitch = TC;
    const int n = g.py, half = n / 2, m = n / Q, logm = ilog2(m), CS = m * TC;
    for (int f = tid; f < (m >> 3) * TC; f += nthr) {
        const int col = f & (TC - 1), b8 = f >> logTC;
        cx<T>* p = s + (b8 * 8) * pitch + col;
        int ro[8];      // rows of the block, cyclically rotated by the block index (see the header)
#pragma unroll
        for (int r = 0; r < 8; r++) ro[r] = ((r + b8) & 7) * pitch;
        cx<T> M[3][8];
#pragma unroll
        for (int c = 0; c < 3; c++) {
#pragma unroll
            for (int r = 0; r < 8; r++) M[c][r] = p[ro[r] + c * CS];
            rad<cx<T>, 8>::fwd(M[c]);
        }
#pragma unroll
        for (int r = 0; r < 8; r++) {
            const int ky = Q * (int)brev((unsigned)(b8 * 8 + r), logm) + q;
            const int kyp = ky <= half ? ky : n - ky;
            const T sy = ky > half ? (T)-1 : (T)1;
            const T* Kp = Kz + (long)kyp * g.Lx + col;
            const T kxx = Kp[0], kyy = Kp[g.kcomp], kzz = Kp[2 * g.kcomp], kxy = sy * Kp[3 * g.kcomp];
            const cx<T> Mx = M[0][r], My = M[1][r], Mz = M[2][r];
            if (IS3D) {
                const T kxz = sz * Kp[4 * g.kcomp], kyz = sy * sz * Kp[5 * g.kcomp];
                M[0][r] = lin3<T>(Mx, -kxx, My, -kxy, Mz, -kxz);
                M[1][r] = lin3<T>(Mx, -kxy, My, -kyy, Mz, -kyz);
                M[2][r] = lin3<T>(Mx, -kxz, My, -kyz, Mz, -kzz);
            } else {
                M[0][r] = lin2<T>(Mx, -kxx, My, -kxy);
                M[1][r] = lin2<T>(Mx, -kxy, My, -kyy);
                M[2][r] = scale<T>(Mz, -kzz);
            }
        }
#pragma unroll
        for (int c = 0; c < 3; c++) {
            rad<cx<T>, 8>::inv(M[c]);
#pragma unroll
            for (int r = 0; r < 8; r++) p[ro[r] + c * CS] = M[c][r];
        }
    }
}

// shared memory (complex elements) of one CTA
MM_HD long smemB4_elems(const Geom& g, int Q) { return (long)(g.py / Q) * 3 * g.TC; }

// phase 1 of CTA q of the cluster of tile `tile`: everything up to z_q in its own tile s.  Requires py/Q >= 16.
template <typename T, int V, int Q>
MM_HD void y_conv_body4_compute(const Geom g, const cx<T>* __restrict__ S, const T* __restrict__ Kh, twiddles<T> tw, cx<T>* s,
                                int tile, int q, int tid, int nthr)
{
    const int ntile = g.Lx / g.TC;
    const int x0 = (tile % ntile) * g.TC, zq = tile / ntile;
    const cx<T>* Sz = S + (long)zq * g.plane + x0;
    const int kz = (int)brev((unsigned)zq, g.logpz);
    const bool is3d = g.nz > 1;
    const int kzp = is3d ? (kz <= g.nz ? kz : g.pz - kz) : 0;
    const T sz = (is3d && kz > g.nz) ? (T)-1 : (T)1;
    const T* Kz = Kh + (long)kzp * g.kplane + x0;
    const int m = g.py / Q, R1 = first_radix(m);
    if (R1 == 8) yB4_first<T, V, 8, Q>(g, Sz, s, tw, q, tid, nthr);
    else if (R1 == 4) yB4_first<T, V, 4, Q>(g, Sz, s, tw, q, tid, nthr);
    else yB4_first<T, V, 2, Q>(g, Sz, s, tw, q, tid, nthr);
    MM_SYNC();
    int Lc = m / R1;
    for (; Lc > 8; Lc >>= 3) { yB4_mid8<T, V, 0>(g, s, m, Lc, tw, tid, nthr); MM_SYNC(); }
    if (is3d) yB4_mul8<T, true, Q>(g, s, Kz, sz, q, tid, nthr);
    else yB4_mul8<T, false, Q>(g, s, Kz, sz, q, tid, nthr);
    MM_SYNC();
    for (Lc = 64; Lc <= m / R1; Lc <<= 3) { yB4_mid8<T, V, 1>(g, s, m, Lc, tw, tid, nthr); MM_SYNC(); }
    if (R1 == 8) yB4_last<T, V, 8, Q>(g, s, tw, q, tid, nthr);
    else if (R1 == 4) yB4_last<T, V, 4, Q>(g, s, tw, q, tid, nthr);
    else yB4_last<T, V, 2, Q>(g, s, tw, q, tid, nthr);
}

// phase 2 of CTA q (after the cluster barrier): rows [q m/Q, (q+1) m/Q) of every block -> finished rows of S.
// tiles[q'] = the tile of CTA q' (own shared memory for q' = q, distributed shared memory otherwise).
template <typename T, int V, int Q>
MM_HD void y_conv_body4_combine(const Geom g, cx<T>* __restrict__ S, cx<T>* const* tiles, int tile, int q, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = TC;
    const int ntile = g.Lx / TC;
    const int x0 = (tile % ntile) * TC, zq = tile / ntile;
    cx<T>* Oz = S + (long)zq * g.plane + x0;
    const int m = g.py / Q, rows = m / Q, i0 = q * rows, CS = m * TC;
    for (int f = tid; f < rows * 3 * LC; f += nthr) {
        const int lc = f & (LC - 1), rest = f >> logLC;
        const int c = rest / rows, i = i0 + rest % rows;
        const int off = c * CS + i * pitch + lc * V;
        E z[Q];
#pragma unroll
        for (int qq = 0; qq < Q; qq++) z[qq] = ldv<E, T>(tiles[qq] + off);
        cx<T>* dst = Oz + (long)c * g.comp + (long)i * g.Lx + lc * V;
        if (Q == 2) {
            stv<E, T>(dst, z[0] + z[1]);
        } else {
            // t = 0: sum; t = 1: weights w_4^(-q') = (+i)^q'
            stv<E, T>(dst, (z[0] + z[2 % Q]) + (z[1] + z[3 % Q]));
            stv<E, T>(dst + (long)m * g.Lx, (z[0] - z[2 % Q]) + mul_pi(z[1] - z[3 % Q]));
        }
    }
}

}  // namespace mm
