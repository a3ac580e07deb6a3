// mm_passB3.cuh — pass B, half-tile form (the long-line path: used when a full py-row tile does not fit one CTA's
// shared memory, e.g. fp64 films of ny >= 4096): the y transform, the spectral multiply and the inverse y transform
// (Eq. 8 in k-space) on HALF tiles.
//
// A zero-padded line of n = 2m points with m non-zero inputs a_i splits, after the folded pad
// stage, into two INDEPENDENT length-m transforms: block 0 = FFT_m(a) holds the even frequencies
// ky = 2q, block 1 = FFT_m(a_i w_n^i) the odd ones ky = 2q+1; multiply and inverse transform stay
// inside a block, and the cropped result is  out_i = r0_i + conj(w_n^i) r1_i.  v3 runs the two
// blocks one after the other through ONE m-row shared-memory tile (half the footprint of v2, so
// two CTAs are resident per SM and one CTA's global loads / stores overlap the other's
// butterflies).  r0 makes a round trip through the output buffer (same thread writes and re-reads
// it, L2-resident); input and output spectra are therefore separate buffers.
//
// Tile element (row p, component c, column col) at s[p*3*TC + c*TC + col]; rows hold bit-reversed
// positions after the forward stages: row p of block ph is frequency ky = 2*brev_m(p) + ph.
#pragma once
#include "mm_fft.cuh"
#include "mm_kernels.cuh"
#include "mm_kernels2.cuh"

namespace mm {

MM_HD void prefetch_l2(const void* p)
{
#if defined(__CUDA_ARCH__)
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
#else
    (void)p;
#endif
}

// first stage of block PH: global load (+ pad twiddle w_n^row for the odd block) + radix R
template <typename T, int V, int R>
MM_HD void yB3_first(const Geom& g, const cx<T>* Sz, cx<T>* s, twiddles<T> tw, int PH, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = 3 * TC;
    const int m = g.ny, n = g.py, sub = m / R;
    for (int f = tid; f < sub * LC; f += nthr) {
        const int lc = f & (LC - 1), i = f >> logLC;
        cx<T> pw[R], wp[R];
        if (R > 1 && i != 0) twiddle_powers<T, R>(tw.get(i, m), pw);
        if (PH) {
#pragma unroll
            for (int r = 0; r < R; r++) wp[r] = tw.get(i + r * sub, n);
        }
#pragma unroll 1
        for (int c = 0; c < 3; c++) {
            const cx<T>* src = Sz + (long)c * g.comp + (long)i * g.Lx + lc * V;
            cx<T>* dst = s + i * pitch + c * TC + lc * V;
            E a[R];
#pragma unroll
            for (int r = 0; r < R; r++) a[r] = ldv<E, T>(src + (long)r * sub * g.Lx);
            if (PH) {
#pragma unroll
                for (int r = 0; r < R; r++) a[r] = cmul(a[r], wp[r]);
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

// last stage of block PH: inverse radix R; block 0 stores r0, block 1 stores r0 + conj(w_n^row) r1
template <typename T, int V, int R>
MM_HD void yB3_last(const Geom& g, cx<T>* Oz, const cx<T>* s, twiddles<T> tw, int PH, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = 3 * TC;
    const int m = g.ny, n = g.py, sub = m / R;
    for (int f = tid; f < sub * LC; f += nthr) {
        const int lc = f & (LC - 1), i = f >> logLC;
        cx<T> pw[R], wp[R];
        if (R > 1 && i != 0) twiddle_powers<T, R>(tw.get(i, m), pw);
        if (PH) {
#pragma unroll
            for (int r = 0; r < R; r++) wp[r] = tw.get(i + r * sub, n);
        }
#pragma unroll 1
        for (int c = 0; c < 3; c++) {
            cx<T>* dstg = Oz + (long)c * g.comp + (long)i * g.Lx + lc * V;
            const cx<T>* src = s + i * pitch + c * TC + lc * V;
            E a[R], r0[R];
            if (PH) {
#pragma unroll
                for (int r = 0; r < R; r++) r0[r] = ldv<E, T>(dstg + (long)r * sub * g.Lx);
            }
#pragma unroll
            for (int r = 0; r < R; r++) a[r] = ldv<E, T>(src + r * sub * pitch);
            if (R > 1 && i != 0) {
#pragma unroll
                for (int r = 1; r < R; r++) a[r] = cmulc(a[r], pw[r]);
            }
            rad<E, R>::inv(a);
#pragma unroll
            for (int r = 0; r < R; r++) stv<E, T>(dstg + (long)r * sub * g.Lx, PH ? r0[r] + cmulc(a[r], wp[r]) : a[r]);
        }
    }
}

// middle radix-8 stage over the m rows of the tile (DIR 0 forward DIF, 1 inverse DIT)
template <typename T, int V, int DIR>
MM_HD void yB3_mid8(const Geom& g, cx<T>* s, int Lc, twiddles<T> tw, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = 3 * TC;
    const int m = g.ny, sub = Lc >> 3, logsub = ilog2(sub);
    for (int f = tid; f < (m >> 3) * LC; f += nthr) {
        const int lc = f & (LC - 1), b = f >> logLC;
        const int blk = b >> logsub, i = b & (sub - 1);
        cx<T> pw[8];
        if (i != 0) twiddle_powers<T, 8>(tw.get(i, Lc), pw);
        cx<T>* base = s + (blk * Lc + i) * pitch + lc * V;
#pragma unroll 1
        for (int c = 0; c < 3; c++) {
            cx<T>* p = base + c * TC;
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

// last forward radix-8 stage (Lc = 8) + multiply by K^ + first inverse stage; three components of
// one column in registers.  Row p of block ph is ky = 2*brev_m(p) + ph.
template <typename T, bool IS3D>
MM_HD void yB3_mul8(const Geom& g, cx<T>* s, const T* Kz, T sz, int ph, int tid, int nthr)
{
    const int TC = g.TC, logTC = ilog2(TC), pitch = 3 * TC;
    const int m = g.ny, n = g.py, logm = g.logny;
    for (int f = tid; f < (m >> 3) * TC; f += nthr) {
        const int col = f & (TC - 1), b8 = f >> logTC;
        cx<T>* p = s + (b8 * 8) * pitch + col;
        cx<T> M[3][8];
#pragma unroll
        for (int c = 0; c < 3; c++) {
#pragma unroll
            for (int r = 0; r < 8; r++) M[c][r] = p[r * pitch + c * TC];
            rad<cx<T>, 8>::fwd(M[c]);
        }
#pragma unroll
        for (int r = 0; r < 8; r++) {
            const int ky = 2 * (int)brev((unsigned)(b8 * 8 + r), logm) + ph;
            const int kyp = ky <= m ? ky : n - ky;
            const T sy = ky > m ? (T)-1 : (T)1;
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
            for (int r = 0; r < 8; r++) p[r * pitch + c * TC] = M[c][r];
        }
    }
}

template <typename T, int V>
MM_HD void yB3_block(const Geom& g, const cx<T>* Sz, cx<T>* Oz, const T* Kz, T sz, twiddles<T> tw, cx<T>* s, int PH, int tid, int nthr)
{
    const int m = g.ny;
    const int R1 = first_radix(m);
    const bool is3d = g.nz > 1;
    // K^ rows of this block (even kyp for block 0, odd for block 1) towards L2 while the FFT runs
    {
        const int ncomp = is3d ? 6 : 4, nrow = (m >> 1) + 1 - PH;
        for (int f = tid; f < nrow * ncomp; f += nthr) {
            const int q = f % ncomp, row = f / ncomp;
            prefetch_l2(Kz + (long)q * g.kcomp + (long)(2 * row + PH) * g.Lx);
        }
    }
    if (R1 == 8) yB3_first<T, V, 8>(g, Sz, s, tw, PH, tid, nthr);
    else if (R1 == 4) yB3_first<T, V, 4>(g, Sz, s, tw, PH, tid, nthr);
    else yB3_first<T, V, 2>(g, Sz, s, tw, PH, tid, nthr);
    MM_SYNC();
    int Lc = m / R1;
    for (; Lc > 8; Lc >>= 3) { yB3_mid8<T, V, 0>(g, s, Lc, tw, tid, nthr); MM_SYNC(); }
    if (is3d) yB3_mul8<T, true>(g, s, Kz, sz, PH, tid, nthr);
    else yB3_mul8<T, false>(g, s, Kz, sz, PH, tid, nthr);
    MM_SYNC();
    for (Lc = 64; Lc <= m / R1; Lc <<= 3) { yB3_mid8<T, V, 1>(g, s, Lc, tw, tid, nthr); MM_SYNC(); }
    if (R1 == 8) yB3_last<T, V, 8>(g, Oz, s, tw, PH, tid, nthr);
    else if (R1 == 4) yB3_last<T, V, 4>(g, Oz, s, tw, PH, tid, nthr);
    else yB3_last<T, V, 2>(g, Oz, s, tw, PH, tid, nthr);
}

// shared memory (complex elements) of pass B v3
MM_HD long smemB3_elems(const Geom& g) { return (long)g.ny * 3 * g.TC; }

// requires ny >= 16 and TC % V == 0.  Sin and Sout must not alias.
template <typename T, int V>
MM_HD void y_conv_body3(const Geom g, const cx<T>* __restrict__ Sin, cx<T>* __restrict__ Sout, const T* __restrict__ Kh,
                        twiddles<T> tw, cx<T>* s, int bid, int tid, int nthr)
{
    const int ntile = g.Lx / g.TC;
    const int x0 = (bid % ntile) * g.TC, zq = bid / ntile;
    const cx<T>* Sz = Sin + (long)zq * g.plane + x0;
    cx<T>* Oz = Sout + (long)zq * g.plane + x0;
    const int kz = (int)brev((unsigned)zq, g.logpz);
    const bool is3d = g.nz > 1;
    const int kzp = is3d ? (kz <= g.nz ? kz : g.pz - kz) : 0;
    const T sz = (is3d && kz > g.nz) ? (T)-1 : (T)1;
    const T* Kz = Kh + (long)kzp * g.kplane + x0;
#pragma unroll 1
    for (int ph = 0; ph < 2; ph++) {
        yB3_block<T, V>(g, Sz, Oz, Kz, sz, tw, s, ph, tid, nthr);
        MM_SYNC();
    }
}

}  // namespace mm
