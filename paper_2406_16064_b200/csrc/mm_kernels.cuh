// mm_kernels.cuh — bodies of the hot-path kernels (demag convolution passes).
//
// Spectrum layout in HBM:  S[c][zpos][j][xpos]  complex, c in {x,y,z}, xpos fastest with row pitch
// Lx >= nx+1.  xpos < nx holds half-spectrum frequency kx = brev(xpos) of the length-2nx real
// transform, xpos == nx holds the Nyquist term; zpos holds kz = brev(zpos); j is a REAL-SPACE row
// index before/after the y pass (the y transform never leaves the SM).  See mm_fft.cuh for why
// everything is kept in bit-reversed positions.
//
//   pass A  fwd_xz   : m, Ms -> S       scale by Ms, pad, R2C along x, pad + FFT along z
//   pass B  y_conv   : S -> S in place  pad + FFT along y, H^ = -K^ M^ (Eq. 8 in k-space,
//                                        PAPER.md:138), inverse FFT along y, crop
//   pass C  inv_zx   : S -> H_d         inverse FFT along z + crop, C2R along x + crop, 1/P
//
// Bodies are __host__ __device__ templates taking (bid, tid, nthr) so the index arithmetic can be
// run on the CPU by a test harness; the __global__ wrappers live in mm_lib.cu.
#pragma once
#include "mm_fft.cuh"

namespace mm {

struct Geom {
    int nx, ny, nz;        // cells
    int px, py, pz;        // padded sizes (2n, or 1 when n == 1)
    int lognx, logny, logpy, logpz;
    int Lx;                // spectrum row pitch in complex elements
    int G;                 // rows (j) per CTA in passes A and C
    int CH;                // x positions per z-chunk in passes A and C (3-D only)
    int TC;                // columns (xpos) per CTA in pass B
    long N;                // nx*ny*nz
    long plane;            // ny * Lx        (one zpos plane of S)
    long comp;             // pz * plane     (one component of S)
    long kplane;           // (ny+1) * Lx    (one kz' plane of K^)
    long kcomp;            // (nz>1 ? nz+1 : 1) * kplane
    int flags;             // tuning bits (MM_FLAGS), 0 = defaults
    int xpad;              // passes A / C (v3 bodies): x tile with one pad point per 8 points and pitch = L (few lines)
};

MM_HD int odd_pitch(int n) { return n | 1; }
// x tile of the v3 passes A / C.  Many lines (L >= 16): pitch L|1, a half-warp covers 16 lines of one point.  Few
// lines (long film lines, L <= 4): the late radix-8 stages would step through the tile with a stride that is a multiple of the
// 32 banks, so point p lives at padded position p + p/8 and the pitch is L itself: a half-warp's 16 (line, butterfly)
// pairs then fall on 32 distinct words at every stage.  ppos is additive over multiples of 8 (all stage strides are).
MM_HD int ppos(int p, int pad) { return pad ? p + (p >> 3) : p; }
MM_HD int x_pitch(const Geom& g) { return g.xpad ? g.G * g.nz : odd_pitch(g.G * g.nz); }
MM_HD long smemA2_elems(const Geom& g) { return (long)(ppos(g.nx, g.xpad) + 1) * x_pitch(g); }

// K^ in the order pass B (v2) consumes it, "Kc": one contiguous tile per (kz', x tile).  The multiply stage
// works on radix-8 blocks b8 of the bit-reversed y spectrum: slot r of block b8 holds ky = brev3(r)*nbk + beta,
// beta = brev(b8), nbk = py/8.  The tensor spectrum is even or odd in ky, and the mirror py - ky of (beta, r) is
// (nbk - beta, 7 - r): blocks pair up, so only the sets beta = 0 .. nbk/2 are stored (half the rows; beta = 0
// and beta = nbk/2 are their own mirrors) and a thread that owns a pair reads one set for both blocks.
// Inside a tile, element (beta, j, col) with j = r*NQ + q (q = tensor component) sits at
// ((beta*NJQ + j/EPL)*TC + col)*EPL + j%EPL, EPL = reals per 16-byte load.  Values are -K^ with the ky mirror
// sign of the odd components (xy, yz) baked in.
MM_HD int kc_nq(const Geom& g) { return g.nz > 1 ? 6 : 4; }
MM_HD long kc_tile_elems(const Geom& g) { return (long)(g.py / 16 + 1) * 8 * kc_nq(g) * g.TC; }
MM_HD long kc_elems(const Geom& g) { return (long)(g.nz > 1 ? g.nz + 1 : 1) * (g.Lx / g.TC) * kc_tile_elems(g); }
template <typename T> MM_HD void kc_fill(const Geom& g, const T* Kh, T* Kc, long idx)
{
    const int NQ = kc_nq(g), EPL = 16 / (int)sizeof(T), NJQ = 8 * NQ / EPL, ntile = g.Lx / g.TC;
    const long tile = kc_tile_elems(g);
    const long t = idx / tile;
    long o = idx - t * tile;
    const int kzp = (int)(t / ntile), xt = (int)(t % ntile);
    const int e = (int)(o % EPL); o /= EPL;
    const int col = (int)(o % g.TC); o /= g.TC;
    const int jq = (int)(o % NJQ), beta = (int)(o / NJQ);
    const int j = jq * EPL + e, q = j % NQ;
    // the set beta = nbk/2 is consumed as the mirror of itself: stored row-reversed with the odd components negated
    const bool self = beta == g.py / 16;
    const int r = self ? 7 - j / NQ : j / NQ;
    const bool odd = q == 3 || q == 5;
    const int ky = (int)brev((unsigned)r, 3) * (g.py / 8) + beta;
    const int kyp = ky <= g.ny ? ky : g.py - ky;
    const T v = Kh[(long)q * g.kcomp + (long)kzp * g.kplane + (long)kyp * g.Lx + xt * g.TC + col];
    const T w = (ky > g.ny && odd) ? v : -v;      // -K^(ky)
    Kc[idx] = (self && odd) ? -w : w;
}

// shared memory (in complex elements) of passes A/C and B
MM_HD long smemA_elems(const Geom& g)
{
    long tile = (long)(g.nx + 1) * odd_pitch(g.G * g.nz);
    long scr = g.nz > 1 ? (long)g.pz * (g.G * g.CH) : 0;
    return tile + scr;
}
MM_HD long smemB_elems(const Geom& g) { return (long)g.py * 3 * g.TC; }

// ------------------------------------------------------------------------------------------------
// Pass A.  One CTA: component c, rows j0..j0+G-1, all z.  grid = 3 * ny/G.
// ------------------------------------------------------------------------------------------------
template <typename T>
MM_HD void fwd_xz_body(const Geom g, const T* __restrict__ m, const T* __restrict__ Ms, cx<T>* __restrict__ S,
                       twiddles<T> tw, cx<T>* smem, int bid, int tid, int nthr)
{
    const int c = bid % 3, j0 = (bid / 3) * g.G;
    const int n = g.nx, h = n / 2, L = g.G * g.nz, pitch = odd_pitch(L);
    cx<T>* s = smem;
    const T* mc = m + (long)c * g.N;
    // load M = Ms m as packed complex pairs; zero-pad stage folded in
    for (int f = tid; f < L * h; f += nthr) {
        const int i = f % h, l = f / h;
        const int gg = l / g.nz, z = l - gg * g.nz;
        const long cell = ((long)z * g.ny + (j0 + gg)) * g.nx + 2 * i;
        const cx<T> mm2 = *reinterpret_cast<const cx<T>*>(mc + cell);
        const cx<T> ms2 = *reinterpret_cast<const cx<T>*>(Ms + cell);
        cx<T> a = mk<T>(ms2.x == (T)0 ? (T)0 : ms2.x * mm2.x, ms2.y == (T)0 ? (T)0 : ms2.y * mm2.y);
        s[(size_t)i * pitch + l] = a;
        s[(size_t)(i + h) * pitch + l] = (i == 0) ? a : cmul(a, tw.get(i, n));
    }
    MM_SYNC();
    fft_fwd_blocks<T>(s, pitch, L, n, h, tw, tid, nthr);
    // real-transform split: X[k] = E[k] + w_{2n}^k O[k] from Z = E + iO
    for (int f = tid; f < L * (h + 1); f += nthr) {
        const int l = f % L, k = f / L;
        if (k == 0) {
            cx<T> z0 = s[l];
            s[l] = mk<T>(z0.x + z0.y, (T)0);
            s[(size_t)n * pitch + l] = mk<T>(z0.x - z0.y, (T)0);
        } else if (k == h) {
            const size_t p = (size_t)brev(k, g.lognx) * pitch + l;
            s[p] = conj(s[p]);
        } else {
            const size_t pa = (size_t)brev(k, g.lognx) * pitch + l, pb = (size_t)brev(n - k, g.lognx) * pitch + l;
            const cx<T> A = s[pa], B = conj(s[pb]);
            const cx<T> E = scale(A + B, (T)0.5), D = scale(A - B, (T)0.5);
            const cx<T> t = cmul(tw.get(k, 2 * n), D);
            s[pa] = E + mul_mi(t);
            s[pb] = conj(E) + mul_mi(conj(t));
        }
    }
    MM_SYNC();
    cx<T>* Sc = S + (long)c * g.comp;
    if (g.nz == 1) {
        for (int f = tid; f < L * (n + 1); f += nthr) {
            const int xp = f % (n + 1), l = f / (n + 1);
            Sc[(long)(j0 + l) * g.Lx + xp] = s[(size_t)xp * pitch + l];
        }
        return;
    }
    // z transform, CH x-positions at a time, through a scratch tile [zq][gg*CH + pl]
    cx<T>* q = smem + (size_t)(n + 1) * pitch;
    const int SL = g.G * g.CH;
    for (int xb = 0; xb < n + 1; xb += g.CH) {
        const int valid = (n + 1 - xb) < g.CH ? (n + 1 - xb) : g.CH;
        for (int f = tid; f < g.nz * SL; f += nthr) {
            const int sl = f % SL, z = f / SL;
            const int gg = sl / g.CH, pl = sl - gg * g.CH;
            cx<T> a = mk<T>((T)0, (T)0);
            if (pl < valid) a = s[(size_t)(xb + pl) * pitch + gg * g.nz + z];
            q[(size_t)z * SL + sl] = a;
            q[(size_t)(z + g.nz) * SL + sl] = (z == 0) ? a : cmul(a, tw.get(z, g.pz));
        }
        MM_SYNC();
        fft_fwd_blocks<T>(q, SL, SL, g.pz, g.nz, tw, tid, nthr);
        for (int f = tid; f < g.pz * SL; f += nthr) {
            const int sl = f % SL, zq = f / SL;
            const int gg = sl / g.CH, pl = sl - gg * g.CH;
            if (pl < valid) Sc[(long)zq * g.plane + (long)(j0 + gg) * g.Lx + xb + pl] = q[(size_t)zq * SL + sl];
        }
        MM_SYNC();
    }
}

// ------------------------------------------------------------------------------------------------
// Pass B.  One CTA: TC columns x0..x0+TC-1 of plane zq, all three components, whole y line.
// grid = (Lx/TC) * pz.   K^ layout: Kh[comp6][kz'][ky'][xpos], real, comp = xx,yy,zz,xy,xz,yz.
// ------------------------------------------------------------------------------------------------
template <typename T>
MM_HD void y_conv_body(const Geom g, cx<T>* __restrict__ S, const T* __restrict__ Kh, twiddles<T> tw, cx<T>* s,
                       int bid, int tid, int nthr)
{
    const int ntile = g.Lx / g.TC;
    const int x0 = (bid % ntile) * g.TC, zq = bid / ntile;
    const int TC = g.TC, L = 3 * TC, pitch = L, ny = g.ny, py = g.py;
    cx<T>* Sz = S + (long)zq * g.plane + x0;
    for (int f = tid; f < ny * L; f += nthr) {
        const int col = f % TC, c = (f / TC) % 3, j = f / L;
        const cx<T> a = Sz[(long)c * g.comp + (long)j * g.Lx + col];
        s[(size_t)j * pitch + c * TC + col] = a;
        s[(size_t)(j + ny) * pitch + c * TC + col] = (j == 0) ? a : cmul(a, tw.get(j, py));
    }
    MM_SYNC();
    fft_fwd_blocks<T>(s, pitch, L, py, ny, tw, tid, nthr);
    // H^_a = - sum_b K^_ab M^_b ; K^ real, symmetric-packed in ky, kz (odd components change sign)
    const int kz = (int)brev((unsigned)zq, g.logpz);
    const bool is3d = g.nz > 1;
    const int kzp = is3d ? (kz <= g.nz ? kz : g.pz - kz) : 0;
    const T sz = (is3d && kz > g.nz) ? (T)-1 : (T)1;
    const T* Kz = Kh + (long)kzp * g.kplane + x0;
    for (int f = tid; f < py * TC; f += nthr) {
        const int col = f % TC, pos = f / TC;
        const int ky = (int)brev((unsigned)pos, g.logpy);
        const int kyp = ky <= ny ? ky : py - ky;
        const T sy = ky > ny ? (T)-1 : (T)1;
        const T* Kp = Kz + (long)kyp * g.Lx + col;
        const T kxx = Kp[0], kyy = Kp[g.kcomp], kzz = Kp[2 * g.kcomp], kxy = sy * Kp[3 * g.kcomp];
        cx<T>* e = s + (size_t)pos * pitch + col;
        const cx<T> Mx = e[0], My = e[TC], Mz = e[2 * TC];
        cx<T> Hx, Hy, Hz;
        if (is3d) {
            const T kxz = sz * Kp[4 * g.kcomp], kyz = sy * sz * Kp[5 * g.kcomp];
            Hx = mk<T>(-(kxx * Mx.x + kxy * My.x + kxz * Mz.x), -(kxx * Mx.y + kxy * My.y + kxz * Mz.y));
            Hy = mk<T>(-(kxy * Mx.x + kyy * My.x + kyz * Mz.x), -(kxy * Mx.y + kyy * My.y + kyz * Mz.y));
            Hz = mk<T>(-(kxz * Mx.x + kyz * My.x + kzz * Mz.x), -(kxz * Mx.y + kyz * My.y + kzz * Mz.y));
        } else {
            Hx = mk<T>(-(kxx * Mx.x + kxy * My.x), -(kxx * Mx.y + kxy * My.y));
            Hy = mk<T>(-(kxy * Mx.x + kyy * My.x), -(kxy * Mx.y + kyy * My.y));
            Hz = mk<T>(-(kzz * Mz.x), -(kzz * Mz.y));
        }
        e[0] = Hx; e[TC] = Hy; e[2 * TC] = Hz;
    }
    MM_SYNC();
    fft_inv_blocks<T>(s, pitch, L, py, ny, tw, tid, nthr);
    for (int f = tid; f < ny * L; f += nthr) {
        const int col = f % TC, c = (f / TC) % 3, j = f / L;
        const size_t p = (size_t)j * pitch + c * TC + col;
        cx<T> a = s[p];
        const cx<T> b = s[p + (size_t)ny * pitch];
        a = (j == 0) ? a + b : a + cmulc(b, tw.get(j, py));
        Sz[(long)c * g.comp + (long)j * g.Lx + col] = a;
    }
}

// ------------------------------------------------------------------------------------------------
// Pass C.  Mirror of pass A: S -> H_d (real space, cropped, scaled by 1/P).  grid = 3 * ny/G.
// ------------------------------------------------------------------------------------------------
template <typename T>
MM_HD void inv_zx_body(const Geom g, const cx<T>* __restrict__ S, T* __restrict__ Hd, twiddles<T> tw, T inv_scale,
                       cx<T>* smem, int bid, int tid, int nthr)
{
    const int c = bid % 3, j0 = (bid / 3) * g.G;
    const int n = g.nx, h = n / 2, L = g.G * g.nz, pitch = odd_pitch(L);
    cx<T>* s = smem;
    const cx<T>* Sc = S + (long)c * g.comp;
    if (g.nz == 1) {
        for (int f = tid; f < L * (n + 1); f += nthr) {
            const int xp = f % (n + 1), l = f / (n + 1);
            s[(size_t)xp * pitch + l] = Sc[(long)(j0 + l) * g.Lx + xp];
        }
        MM_SYNC();
    } else {
        cx<T>* q = smem + (size_t)(n + 1) * pitch;
        const int SL = g.G * g.CH;
        for (int xb = 0; xb < n + 1; xb += g.CH) {
            const int valid = (n + 1 - xb) < g.CH ? (n + 1 - xb) : g.CH;
            for (int f = tid; f < g.pz * SL; f += nthr) {
                const int sl = f % SL, zq = f / SL;
                const int gg = sl / g.CH, pl = sl - gg * g.CH;
                cx<T> a = mk<T>((T)0, (T)0);
                if (pl < valid) a = Sc[(long)zq * g.plane + (long)(j0 + gg) * g.Lx + xb + pl];
                q[(size_t)zq * SL + sl] = a;
            }
            MM_SYNC();
            fft_inv_blocks<T>(q, SL, SL, g.pz, g.nz, tw, tid, nthr);
            for (int f = tid; f < g.nz * SL; f += nthr) {
                const int sl = f % SL, z = f / SL;
                const int gg = sl / g.CH, pl = sl - gg * g.CH;
                if (pl >= valid) continue;
                cx<T> a = q[(size_t)z * SL + sl];
                const cx<T> b = q[(size_t)(z + g.nz) * SL + sl];
                a = (z == 0) ? a + b : a + cmulc(b, tw.get(z, g.pz));
                s[(size_t)(xb + pl) * pitch + gg * g.nz + z] = a;
            }
            MM_SYNC();
        }
    }
    // merge: Z'[k] = 2 Z[k] = (X[k] + conj X[n-k]) + i conj(w_{2n}^k) (X[k] - conj X[n-k])
    for (int f = tid; f < L * (h + 1); f += nthr) {
        const int l = f % L, k = f / L;
        if (k == 0) {
            const cx<T> A = s[l], B = conj(s[(size_t)n * pitch + l]);
            s[l] = (A + B) + mul_pi(A - B);
        } else if (k == h) {
            const size_t p = (size_t)brev(k, g.lognx) * pitch + l;
            s[p] = scale(conj(s[p]), (T)2);
        } else {
            const size_t pa = (size_t)brev(k, g.lognx) * pitch + l, pb = (size_t)brev(n - k, g.lognx) * pitch + l;
            const cx<T> A = s[pa], B = conj(s[pb]);
            const cx<T> E = A + B, O = cmulc(A - B, tw.get(k, 2 * n));
            s[pa] = E + mul_pi(O);
            s[pb] = conj(E) + mul_pi(conj(O));
        }
    }
    MM_SYNC();
    fft_inv_blocks<T>(s, pitch, L, n, h, tw, tid, nthr);
    T* Hc = Hd + (long)c * g.N;
    for (int f = tid; f < L * h; f += nthr) {
        const int i = f % h, l = f / h;
        const int gg = l / g.nz, z = l - gg * g.nz;
        cx<T> a = s[(size_t)i * pitch + l];
        const cx<T> b = s[(size_t)(i + h) * pitch + l];
        a = (i == 0) ? a + b : a + cmulc(b, tw.get(i, n));
        const long cell = ((long)z * g.ny + (j0 + gg)) * g.nx + 2 * i;
        *reinterpret_cast<cx<T>*>(Hc + cell) = scale(a, inv_scale);
    }
}

}  // namespace mm
