// mm_passAC.cuh — v3 bodies of passes A (fwd_xz) and C (inv_zx): same math and memory layout as
// mm_kernels2.cuh, restructured around what the profiles showed (profiles/r01_*): the x tile is
// not bandwidth bound, it is bound by integer / control instructions and by bank conflicts.
//   * middle radix-8 stages: the LINE index is the fastest lane index (a half-warp touches 16
//     consecutive lines = one 128-byte row: conflict-free at every stage), each thread runs TB
//     blocks that share one twiddle set, all loops have compile-time trip counts;
//   * pass A: the real-transform split X[k] = E[k] - i w_2n^k D[k] (pairs k, n-k) is done by the
//     consumer, the register z transform, which reads its own position and the partner position
//     from the tile — the separate split sweep over the tile (a full shared-memory round trip, a
//     barrier and ~1/3 of the pass's instructions) is gone; the twiddle and the index arithmetic
//     are shared by the nz values of one thread.
#pragma once
#include "mm_fft.cuh"
#include "mm_kernels.cuh"
#include "mm_kernels2.cuh"

namespace mm {

// radix-8 stage on blocks of length Lc of n-point lines; lanes run over lines, TB blocks per thread
template <typename T, int DIR, int TB, bool PAD>
MM_HD void xs_mid8b(cx<T>* s, int pitch, int L, int n, int Lc, twiddles<T> tw, int tid, int nthr)
{
    constexpr int pad = PAD ? 1 : 0;
    const int logL = ilog2(L), sub = Lc >> 3, logsub = ilog2(sub);
    const int stride = ppos(sub, pad) * pitch, bstride = ppos(Lc, pad) * pitch;
    const int nitem = L * sub * ((n / Lc) / TB);
    for (int f = tid; f < nitem; f += nthr) {
        const int l = f & (L - 1), rest = f >> logL;
        const int i = rest & (sub - 1), bg = rest >> logsub;
        cx<T> pw[8];
        if (i != 0) twiddle_powers<T, 8>(tw.get(i, Lc), pw);
        cx<T>* p = s + (bg * TB * ppos(Lc, pad) + ppos(i, pad)) * pitch + l;
#pragma unroll
        for (int t = 0; t < TB; t++, p += bstride) {
            cx<T> v[8];
#pragma unroll
            for (int r = 0; r < 8; r++) v[r] = p[r * stride];
            if (DIR == 0) {
                rad<cx<T>, 8>::fwd(v);
                if (i != 0) {
#pragma unroll
                    for (int r = 1; r < 8; r++) v[r] = cmul(v[r], pw[r]);
                }
            } else {
                if (i != 0) {
#pragma unroll
                    for (int r = 1; r < 8; r++) v[r] = cmulc(v[r], pw[r]);
                }
                rad<cx<T>, 8>::inv(v);
            }
#pragma unroll
            for (int r = 0; r < 8; r++) p[r * stride] = v[r];
        }
    }
}

template <typename T, int DIR, bool PAD>
MM_HD void xs_mid8_any(cx<T>* s, int pitch, int L, int n, int Lc, twiddles<T> tw, int tid, int nthr)
{
    const int nblk = n / Lc;
    if (nblk % 4 == 0) xs_mid8b<T, DIR, 4, PAD>(s, pitch, L, n, Lc, tw, tid, nthr);
    else if (nblk % 2 == 0) xs_mid8b<T, DIR, 2, PAD>(s, pitch, L, n, Lc, tw, tid, nthr);
    else xs_mid8b<T, DIR, 1, PAD>(s, pitch, L, n, Lc, tw, tid, nthr);
}

// padded z transform of the NZ values a[] of one (row, x position) and store to S (NZ = 1: plain store)
template <typename T, int NZ>
MM_HD void zfft_store(const Geom& g, cx<T>* dst, cx<T>* a, twiddles<T> tw)
{
    if (NZ == 1) { dst[0] = a[0]; return; }
    {
        cx<T> v[NZ];
#pragma unroll
        for (int z = 0; z < NZ; z++) v[z] = a[z];
        rad<cx<T>, NZ>::fwd(v);
#pragma unroll
        for (int z = 0; z < NZ; z++) dst[(long)z * g.plane] = v[z];
    }
#pragma unroll
    for (int z = 1; z < NZ; z++) a[z] = rot_w<T, 2 * NZ>(a[z], z);      // * w_2NZ^z, an immediate
    rad<cx<T>, NZ>::fwd(a);
#pragma unroll
    for (int z = 0; z < NZ; z++) dst[(long)(NZ + z) * g.plane] = a[z];
}

// Pass A tail: split of the packed real transform fused into the register z transform.
// Tile s holds Z (the n-point complex transform of the packed pairs) in bit-reversed positions;
// thread (xp, gg) forms X[k], k = brev(xp), from Z at xp and at the partner position brev(n-k):
//   X[k] = (Z[k] + conj Z[n-k])/2 - i w_2n^k (Z[k] - conj Z[n-k])/2 ,  X[0] = Re Z0 + Im Z0,
// and X[n] = Re Z0 - Im Z0 (stored at xpos = n).
template <typename T, int NZ, bool PAD>
MM_HD void zA_split_regs(const Geom& g, cx<T>* Sc, const cx<T>* s, int pitch, int j0, twiddles<T> tw, int tid, int nthr)
{
    const int n = g.nx, lognx = g.lognx;
    for (int f = tid; f < n * g.G; f += nthr) {
        const int xp = f & (n - 1), gg = f >> lognx;
        const int k = (int)brev((unsigned)xp, lognx);
        const cx<T>* pa = s + ppos(xp, PAD) * pitch + gg * NZ;
        cx<T> a[NZ];
        if (k == 0) {
#pragma unroll
            for (int z = 0; z < NZ; z++) { const cx<T> z0 = pa[z]; a[z] = mk<T>(z0.x + z0.y, (T)0); }
        } else {
            const cx<T>* pb = s + ppos((int)brev((unsigned)(n - k), lognx), PAD) * pitch + gg * NZ;
            const cx<T> w = tw.get(k, 2 * n);
            const cx<T> w2 = mk<T>((T)0.5 * w.y, (T)-0.5 * w.x);      // -i w / 2
#pragma unroll
            for (int z = 0; z < NZ; z++) {
                const cx<T> A = pa[z], B = conj(pb[z]);
                const cx<T> t = cmul(A - B, w2);
                a[z] = scale(A + B, (T)0.5) + t;
            }
        }
        zfft_store<T, NZ>(g, Sc + (long)(j0 + gg) * g.Lx + xp, a, tw);
    }
    for (int gg = tid; gg < g.G; gg += nthr) {      // Nyquist column
        const cx<T>* pa = s + gg * NZ;
        cx<T> a[NZ];
#pragma unroll
        for (int z = 0; z < NZ; z++) { const cx<T> z0 = pa[z]; a[z] = mk<T>(z0.x - z0.y, (T)0); }
        zfft_store<T, NZ>(g, Sc + (long)(j0 + gg) * g.Lx + n, a, tw);
    }
}

// requires nx >= 32, NZ in {1,2,4,8,16,32}
template <typename T, int NZ, bool PAD = false>
MM_HD void fwd_xz_body3(const Geom g, const T* __restrict__ mvec, const T* __restrict__ Ms, cx<T>* __restrict__ S,
                        twiddles<T> tw, cx<T>* s, int bid, int tid, int nthr)
{
    const int c = bid % 3, j0 = (bid / 3) * g.G;
    const int n = g.nx, m = n / 2, L = g.G * g.nz, pitch = PAD ? L : odd_pitch(L);
    const T* mc = mvec + (long)c * g.N;
    const int R1 = first_radix(m);
    if (R1 == 8) xA_first<T, 8, PAD>(g, mc, Ms, s, pitch, j0, tw, tid, nthr);
    else if (R1 == 4) xA_first<T, 4, PAD>(g, mc, Ms, s, pitch, j0, tw, tid, nthr);
    else xA_first<T, 2, PAD>(g, mc, Ms, s, pitch, j0, tw, tid, nthr);
    MM_SYNC();
    for (int Lc = m / R1; Lc > 1; Lc >>= 3) { xs_mid8_any<T, 0, PAD>(s, pitch, L, n, Lc, tw, tid, nthr); MM_SYNC(); }
    zA_split_regs<T, NZ, PAD>(g, S + (long)c * g.comp, s, pitch, j0, tw, tid, nthr);
}

// Pass C head: merge of the packed real transform (pairs k, n-k) fused with the first inverse radix-8
// stage (Lc = 8).  Position p = blk*8 + r holds k = brev3(r)*nb + beta, beta = brev(blk), nb = n/8; the
// partner n-k sits at r' = 7-r of block blk' = brev(nb - beta): blocks pair up, so one thread merges
// and transforms BOTH blocks of a pair in place (no cross-thread hazard, no separate merge sweep):
//   Z'[k] = (X[k] + conj X[n-k]) + i conj(w_2n^k) (X[k] - conj X[n-k]),  Z'[n-k] = conj(E) + i conj(O);
//   Z'[0] = (X[0] + conj X[n]) + i (X[0] - conj X[n])   (X[n] is stored at position n).
template <typename T, bool PAD>
MM_HD void xC_merge8(const Geom& g, cx<T>* s, int pitch, int L, twiddles<T> tw, int tid, int nthr)
{
    const int n = g.nx, nb = n >> 3, logb = g.lognx - 3, logL = ilog2(L);
    for (int f = tid; f < (nb / 2 + 1) * L; f += nthr) {
        const int l = f & (L - 1), beta = f >> logL;
        cx<T>* pA = s + ppos((int)brev((unsigned)beta, logb) * 8, PAD) * pitch + l;
        cx<T> w[8];
#pragma unroll
        for (int r = 0; r < 8; r++) w[r] = tw.get((int)brev((unsigned)r, 3) * nb + beta, 2 * n);
        cx<T> ZA[8];
#pragma unroll
        for (int r = 0; r < 8; r++) ZA[r] = pA[r * pitch];
        if (beta != 0 && beta != nb / 2) {
            cx<T>* pB = s + ppos((int)brev((unsigned)(nb - beta), logb) * 8, PAD) * pitch + l;
            cx<T> ZB[8];
#pragma unroll
            for (int r = 0; r < 8; r++) ZB[r] = pB[r * pitch];
#pragma unroll
            for (int r = 0; r < 8; r++) {
                const cx<T> A = ZA[r], B = conj(ZB[7 - r]);
                const cx<T> E = A + B, O = cmulc(A - B, w[r]);
                ZA[r] = E + mul_pi(O);
                ZB[7 - r] = conj(E) + mul_pi(conj(O));
            }
            rad<cx<T>, 8>::inv(ZB);
#pragma unroll
            for (int r = 0; r < 8; r++) pB[r * pitch] = ZB[r];
        } else if (beta != 0) {      // self-paired block: r <-> 7-r
#pragma unroll
            for (int r = 0; r < 4; r++) {
                const cx<T> A = ZA[r], B = conj(ZA[7 - r]);
                const cx<T> E = A + B, O = cmulc(A - B, w[r]);
                ZA[r] = E + mul_pi(O);
                ZA[7 - r] = conj(E) + mul_pi(conj(O));
            }
        } else {                     // block 0: k = rho*nb; r=0 <-> Nyquist slot, r=1 is k = n/2, pairs (4,7) (2,3) (6,5)
            {
                const cx<T> A = ZA[0], B = conj(s[ppos(n, PAD) * pitch + l]);
                ZA[0] = (A + B) + mul_pi(A - B);
            }
            ZA[1] = scale(conj(ZA[1]), (T)2);
            const int ra[3] = { 4, 2, 6 }, rb[3] = { 7, 3, 5 };
#pragma unroll
            for (int q = 0; q < 3; q++) {
                const cx<T> A = ZA[ra[q]], B = conj(ZA[rb[q]]);
                const cx<T> E = A + B, O = cmulc(A - B, w[ra[q]]);
                ZA[ra[q]] = E + mul_pi(O);
                ZA[rb[q]] = conj(E) + mul_pi(conj(O));
            }
        }
        rad<cx<T>, 8>::inv(ZA);
#pragma unroll
        for (int r = 0; r < 8; r++) pA[r * pitch] = ZA[r];
    }
}

template <typename T, int NZ, bool PAD = false>
MM_HD void inv_zx_body3(const Geom g, const cx<T>* __restrict__ S, T* __restrict__ Hd, twiddles<T> tw, T inv_scale,
                        cx<T>* s, int bid, int tid, int nthr)
{
    const int c = bid % 3, j0 = (bid / 3) * g.G;
    const int n = g.nx, m = n / 2, L = g.G * g.nz, pitch = PAD ? L : odd_pitch(L);
    const cx<T>* Sc = S + (long)c * g.comp;
    if (NZ == 1) {
        for (int f = tid; f < L * (n + 1); f += nthr) {
            const int xp = f % (n + 1), l = f / (n + 1);
            s[ppos(xp, PAD) * pitch + l] = Sc[(long)(j0 + l) * g.Lx + xp];
        }
    } else {
        zC_regs<T, NZ, PAD>(g, Sc, s, pitch, j0, tw, tid, nthr);
    }
    MM_SYNC();
    xC_merge8<T, PAD>(g, s, pitch, L, tw, tid, nthr);
    MM_SYNC();
    const int R1 = first_radix(m);
    for (int Lc = 64; Lc <= m / R1; Lc <<= 3) { xs_mid8_any<T, 1, PAD>(s, pitch, L, n, Lc, tw, tid, nthr); MM_SYNC(); }
    T* Hc = Hd + (long)c * g.N;
    if (R1 == 8) xC_last<T, 8, PAD>(g, Hc, s, pitch, j0, inv_scale, tw, tid, nthr);
    else if (R1 == 4) xC_last<T, 4, PAD>(g, Hc, s, pitch, j0, inv_scale, tw, tid, nthr);
    else xC_last<T, 2, PAD>(g, Hc, s, pitch, j0, inv_scale, tw, tid, nthr);
}

}  // namespace mm
