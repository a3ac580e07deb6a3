// mm_passB7.cuh — pass B (pad + FFT y, H^ = -K^ M^ of Eq. 8 in k-space, inverse FFT y, crop)
// specialised at compile time: ny = 2^LOGM, TC = 2^LOGTC columns of 32 bytes per row (fp32: TC = 4, 256 threads;
// fp64: TC = 2, 128 threads with twice the registers), component-major tile moved by TMA box copies.  Same math, tile layout and K^ layout ("Kc", mm_kernels.cuh) as y_conv_body5 in
// mm_kernels2.cuh; what changes is how the work is issued (profiles/r02_*: the generic body spends a quarter
// of its warp time on exposed global-load latency and on index arithmetic):
//   * every stride and trip count is a constant, so the shared-memory accesses of a stage are base + immediate
//     and there is no division, no loop bookkeeping (one item per thread per stage when ny = 512);
//   * the twiddle of the NEXT stage (one table value per thread; the radix powers and the pad / crop twiddles
//     are derived from it) and the K^ set of the multiply stage are loaded BEFORE the block barrier that ends
//     the previous stage, so their latency is covered by the barrier wait instead of heading the next stage;
//   * the first stage's twiddles are formed while the TMA loads of the tile are in flight.
// Everything is __host__ __device__ (NTHR = 256 on the device, where every stage has at most one item per
// thread and the item loops fold away; tid = 0, NTHR = 1 on the CPU, where the prefetched values are
// recomputed per item) so tests/host_emul can check the index arithmetic without a GPU.
#pragma once
#include "mm_fft.cuh"
#include "mm_kernels.cuh"
#include "mm_kernels2.cuh"

namespace mm {

template <int LOGM, int LOGTC> struct B7 {
    static constexpr int M = 1 << LOGM, N = 2 * M, TC = 1 << LOGTC;
    static constexpr int R1 = (LOGM % 3 == 0) ? 8 : ((LOGM % 3 == 2) ? 4 : 2);      // first_radix(M)
    static constexpr int LOGR1 = (LOGM % 3 == 0) ? 3 : (LOGM % 3);
    static constexpr int SUB1 = M / R1;                 // butterflies of the first / last stage per column
    static constexpr int CS = N * TC;                   // component stride of the tile (complex elements)
    static constexpr int NBK = N / 8;                   // radix-8 blocks of the multiply stage
    static constexpr int RB = M < 256 ? M : 256;        // rows per TMA box
    static_assert(LOGM >= 4 && LOGTC >= 1, "ny >= 16, TC >= 2");
};

template <typename T> struct tw8 { cx<T> p[8]; };      // p[r] = w^brev3(r), p[0] unused

// twiddle set of a radix-8 stage on blocks of length Lc (butterfly i): powers of w_Lc^i
template <typename T> MM_HD tw8<T> b7_mid_tw(twiddles<T> tw, int logtw, int logLc, int i)
{
    tw8<T> r;
    twiddle_powers<T, 8>(tw.tw[i << (logtw - logLc)], r.p);
    return r;
}

template <typename T, int R> struct twfl { cx<T> wp[R], pw[R]; };
// first / last stage: pad (crop) twiddles w_n^(i + r sub) and the radix-R powers of w_m^i = (w_n^i)^2
template <typename T, int R> MM_HD twfl<T, R> b7_fl_tw(twiddles<T> tw, int logtw, int logn, int i)
{
    twfl<T, R> r;
    pad_twiddles<T, R>(tw.tw[i << (logtw - logn)], r.wp);
    r.pw[0] = mk<T>((T)1, (T)0);
    if (R > 1) twiddle_powers<T, R>(cmul(r.wp[0], r.wp[0]), r.pw);
    return r;
}

// ---- stages ------------------------------------------------------------------------------------------------
// first: rows i + r*SUB1 of the TMA-deposited lower half -> radix R1 of (a) and of (a * pad twiddle), both halves
template <int LOGM, int LOGTC, int NTHR, typename T>
MM_HD void b7_first(cx<T>* s, const twfl<T, B7<LOGM, LOGTC>::R1>& pre, twiddles<T> tw, int logtw, int tid, int nthr, unsigned long long* bars)
{
    typedef B7<LOGM, LOGTC> P;
    constexpr int R = P::R1, TC = P::TC;
    bool first = true;
    for (int f = tid; f < P::SUB1 * TC; f += NTHR, first = false) {
        const int col = f & (TC - 1), i = f >> LOGTC;
        const twfl<T, R> t = first ? pre : b7_fl_tw<T, R>(tw, logtw, LOGM + 1, i);
        cx<T>* base = s + i * TC + col;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            cx<T>* p = base + c * P::CS;
            if (bars != nullptr) mbar_wait0(bars + c);
            cx<T> a[R], u[R];
#pragma unroll
            for (int r = 0; r < R; r++) a[r] = p[r * P::SUB1 * TC];
#pragma unroll
            for (int r = 0; r < R; r++) u[r] = cmul(a[r], t.wp[r]);
            rad<cx<T>, R>::fwd(a);
            rad<cx<T>, R>::fwd(u);
#pragma unroll
            for (int r = 1; r < R; r++) { a[r] = cmul(a[r], t.pw[r]); u[r] = cmul(u[r], t.pw[r]); }
#pragma unroll
            for (int r = 0; r < R; r++) { p[r * P::SUB1 * TC] = a[r]; p[(P::M + r * P::SUB1) * TC] = u[r]; }
        }
    }
}

// last: inverse radix R1 on both halves, crop combine a + conj(w) u -> the lower half of the tile
template <int LOGM, int LOGTC, int NTHR, typename T>
MM_HD void b7_last(cx<T>* s, const twfl<T, B7<LOGM, LOGTC>::R1>& pre, twiddles<T> tw, int logtw, int tid, int nthr)
{
    typedef B7<LOGM, LOGTC> P;
    constexpr int R = P::R1, TC = P::TC;
    bool first = true;
    for (int f = tid; f < P::SUB1 * TC; f += NTHR, first = false) {
        const int col = f & (TC - 1), i = f >> LOGTC;
        const twfl<T, R> t = first ? pre : b7_fl_tw<T, R>(tw, logtw, LOGM + 1, i);
        cx<T>* base = s + i * TC + col;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            cx<T>* p = base + c * P::CS;
            cx<T> a[R], u[R];
#pragma unroll
            for (int r = 0; r < R; r++) { a[r] = p[r * P::SUB1 * TC]; u[r] = p[(P::M + r * P::SUB1) * TC]; }
#pragma unroll
            for (int r = 1; r < R; r++) { a[r] = cmulc(a[r], t.pw[r]); u[r] = cmulc(u[r], t.pw[r]); }
            rad<cx<T>, R>::inv(a);
            rad<cx<T>, R>::inv(u);
#pragma unroll
            for (int r = 0; r < R; r++) p[r * P::SUB1 * TC] = a[r] + cmulc(u[r], t.wp[r]);
        }
    }
}

// middle radix-8 stage on blocks of length 2^LOGLC, 16 bytes per shared-memory access (fp32: two columns, fp64: one —
// the lanes of a warp then cover consecutive 16-byte words: conflict-free in both precisions)
template <typename T> struct b7_v { static constexpr int LOGV = sizeof(T) == 8 ? 0 : 1, V = 1 << LOGV; };
template <int LOGM, int LOGTC, int LOGLC, int DIR, int NTHR, typename T>
MM_HD void b7_mid8(cx<T>* s, const tw8<T>& pre, twiddles<T> tw, int logtw, int tid, int nthr)
{
    typedef B7<LOGM, LOGTC> P;
    constexpr int V = b7_v<T>::V, LOGLCV = LOGTC - b7_v<T>::LOGV, LCV = 1 << LOGLCV;
    typedef cvec<T, V> E;
    constexpr int TC = P::TC, SUB = 1 << (LOGLC - 3), RS = SUB * TC;
    bool first = true;
    for (int f = tid; f < (P::N >> 3) * LCV; f += NTHR, first = false) {
        const int lc = f & (LCV - 1), b = f >> LOGLCV;
        const int blk = b >> (LOGLC - 3), i = b & (SUB - 1);
        const tw8<T> t = first ? pre : b7_mid_tw<T>(tw, logtw, LOGLC, i);
        cx<T>* base = s + ((blk << LOGLC) + i) * TC + lc * V;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            cx<T>* p = base + c * P::CS;
            E v[8];
#pragma unroll
            for (int r = 0; r < 8; r++) v[r] = ldv<E, T>(p + r * RS);
            if (DIR == 0) {
                rad<E, 8>::fwd(v);
#pragma unroll
                for (int r = 1; r < 8; r++) v[r] = cmul(v[r], t.p[r]);
            } else {
#pragma unroll
                for (int r = 1; r < 8; r++) v[r] = cmulc(v[r], t.p[r]);
                rad<E, 8>::inv(v);
            }
#pragma unroll
            for (int r = 0; r < 8; r++) stv<E, T>(p + r * RS, v[r]);
        }
    }
}
template <int LOGTC, typename T> MM_HD int b7_mid_i(int f, int logLc) { return (f >> (LOGTC - b7_v<T>::LOGV)) & ((1 << (logLc - 3)) - 1); }

template <typename T, int NJ> struct kset { T k[NJ]; };
// 16-byte loads jq in [JQ0, JQ1) of the K^ set `set` of column `col` into r (the whole set: JQ0 = 0, JQ1 = NJQ)
template <typename T, bool IS3D, int TC, int JQ0, int JQ1> MM_HD void b7_kload_part(const T* Kt, int set, int col, kset<T, IS3D ? 48 : 32>& r)
{
    constexpr int NQ = IS3D ? 6 : 4, NJ = 8 * NQ, EPL = 16 / (int)sizeof(T);
    const T* Kp = Kt + (long)set * (NJ * TC) + col * EPL;
#pragma unroll
    for (int jq = JQ0; jq < JQ1; jq++) {
        const kvec<T> v = *reinterpret_cast<const kvec<T>*>(Kp + jq * TC * EPL);
#pragma unroll
        for (int e = 0; e < EPL; e++) r.k[jq * EPL + e] = v.e[e];
    }
}
template <typename T, bool IS3D, int TC> MM_HD kset<T, IS3D ? 48 : 32> b7_kload(const T* Kt, int set, int col)
{
    constexpr int NJQ = 8 * (IS3D ? 6 : 4) / (16 / (int)sizeof(T));
    kset<T, IS3D ? 48 : 32> r;
    b7_kload_part<T, IS3D, TC, 0, NJQ>(Kt, set, col, r);
    return r;
}
// how much of the first multiply item's K^ set is loaded BEFORE the barrier that precedes the multiply stage (its
// latency hides under the barrier wait); the rest is loaded right after the barrier and hides under the three 8-point
// transforms.  3-D: one third (MM_B7_PRE3 = 1).  Measured on cfg4 fp32 (profiles/r02_experiments.md): the whole set
// (48 registers) across the barrier spilled 9 registers whose spill stores waited for the loads — 193.2 us; one third
// 186.4 us; nothing before the barrier 191.3 us.
#ifndef MM_B7_PRE3
#define MM_B7_PRE3 1
#endif
template <typename T, bool IS3D> struct B7Pre { static constexpr int NJQ = 8 * (IS3D ? 6 : 4) / (16 / (int)sizeof(T)), PRE = IS3D ? (MM_B7_PRE3 * NJQ) / 3 : NJQ; };

// multiply stage: item = (column, mirror pair of 8-row blocks), see yB_mul8 in mm_kernels2.cuh
template <int LOGM, int LOGTC, bool IS3D, int NTHR, typename T>
MM_HD void b7_mul8(cx<T>* s, const kset<T, IS3D ? 48 : 32>& pre, const T* Kt, T sz, int tid, int nthr)
{
    typedef B7<LOGM, LOGTC> P;
    constexpr int NQ = IS3D ? 6 : 4, NJ = 8 * NQ, TC = P::TC, NBK = P::NBK, LOGNBK = LOGM - 2;
    bool first = true;
    for (int f = tid; f < (NBK >> 1) * TC; f += NTHR, first = false) {
        const int col = f & (TC - 1), t = f >> LOGTC;
        kset<T, NJ> K;
        if (first) { K = pre; b7_kload_part<T, IS3D, TC, B7Pre<T, IS3D>::PRE, B7Pre<T, IS3D>::NJQ>(Kt, t, col, K); }
        else K = b7_kload<T, IS3D, TC>(Kt, t, col);
        int ro[8];
#pragma unroll
        for (int r = 0; r < 8; r++) ro[r] = ((r + t) & 7) * TC;
#pragma unroll
        for (int h = 0; h < 2; h++) {
            const int beta = h == 0 ? t : (t == 0 ? (NBK >> 1) : NBK - t);
            if (h == 1 && t == 0) K = b7_kload<T, IS3D, TC>(Kt, NBK >> 1, col);
            cx<T>* p = s + ((int)brev((unsigned)beta, LOGNBK) * 8) * TC + col;
            cx<T> Mv[3][8];
#pragma unroll
            for (int c = 0; c < 3; c++) {
#pragma unroll
                for (int r = 0; r < 8; r++) Mv[c][r] = p[ro[r] + c * P::CS];
                rad<cx<T>, 8>::fwd(Mv[c]);
            }
#pragma unroll
            for (int r = 0; r < 8; r++) {
                const int kr = (h == 0 ? r : 7 - r) * NQ;
                const T so = h == 0 ? (T)1 : (T)-1;
                const T kxx = K.k[kr], kyy = K.k[kr + 1], kzz = K.k[kr + 2], kxy = so * K.k[kr + 3];
                const cx<T> Mx = Mv[0][r], My = Mv[1][r], Mz = Mv[2][r];
                if (IS3D) {
                    const T kxz = sz * K.k[kr + (IS3D ? 4 : 0)], kyz = (so * sz) * K.k[kr + (IS3D ? 5 : 0)];
                    Mv[0][r] = lin3<T>(Mx, kxx, My, kxy, Mz, kxz);
                    Mv[1][r] = lin3<T>(Mx, kxy, My, kyy, Mz, kyz);
                    Mv[2][r] = lin3<T>(Mx, kxz, My, kyz, Mz, kzz);
                } else {
                    Mv[0][r] = lin2<T>(Mx, kxx, My, kxy);
                    Mv[1][r] = lin2<T>(Mx, kxy, My, kyy);
                    Mv[2][r] = scale<T>(Mz, kzz);
                }
            }
#pragma unroll
            for (int c = 0; c < 3; c++) {
                rad<cx<T>, 8>::inv(Mv[c]);
#pragma unroll
                for (int r = 0; r < 8; r++) p[ro[r] + c * P::CS] = Mv[c][r];
            }
        }
    }
}

// forward middle stages Lc = 2^LOGLC, 2^(LOGLC-3), ..., 64 ; each one ends with the block barrier and, before
// it, the loads of what the following stage needs first (its twiddle; the K^ set of the multiply stage)
template <int LOGM, int LOGTC, int LOGLC, bool IS3D, int NTHR, typename T>
MM_HD void b7_fwd_mids(cx<T>* s, twiddles<T> tw, int logtw, const T* Kt, int tid, int nthr, kset<T, IS3D ? 48 : 32>& kpre)
{
    if constexpr (LOGLC > 3) {
        const tw8<T> t = b7_mid_tw<T>(tw, logtw, LOGLC, b7_mid_i<LOGTC, T>(tid, LOGLC));
        MM_SYNC();
        b7_mid8<LOGM, LOGTC, LOGLC, 0, NTHR, T>(s, t, tw, logtw, tid, nthr);
        b7_fwd_mids<LOGM, LOGTC, LOGLC - 3, IS3D, NTHR, T>(s, tw, logtw, Kt, tid, nthr, kpre);
    } else {
        if (tid < (B7<LOGM, LOGTC>::NBK >> 1) * B7<LOGM, LOGTC>::TC)      // K^ set of the thread's first multiply item (the part that fits in registers)
            b7_kload_part<T, IS3D, B7<LOGM, LOGTC>::TC, 0, B7Pre<T, IS3D>::PRE>(Kt, tid >> LOGTC, tid & (B7<LOGM, LOGTC>::TC - 1), kpre);
        MM_SYNC();
    }
}
// inverse middle stages Lc = 2^LOGLC, ..., 2^LOGTOP
template <int LOGM, int LOGTC, int LOGLC, int LOGTOP, int NTHR, typename T>
MM_HD void b7_inv_mids(cx<T>* s, twiddles<T> tw, int logtw, int tid, int nthr)
{
    if constexpr (LOGLC <= LOGTOP) {
        const tw8<T> t = b7_mid_tw<T>(tw, logtw, LOGLC, b7_mid_i<LOGTC, T>(tid, LOGLC));
        MM_SYNC();
        b7_mid8<LOGM, LOGTC, LOGLC, 1, NTHR, T>(s, t, tw, logtw, tid, nthr);
        b7_inv_mids<LOGM, LOGTC, LOGLC + 3, LOGTOP, NTHR, T>(s, tw, logtw, tid, nthr);
    }
}

// One tile.  `tmap` = CUtensorMap of S as (x, j, zpos, comp); `bar` = three 8-byte shared-memory mbarriers.
template <int LOGM, int LOGTC, bool IS3D, int NTHR, typename T>
MM_HD void y_conv_body7(const Geom g, cx<T>* __restrict__ S, const T* __restrict__ Kc, twiddles<T> tw, int logtw, cx<T>* s,
                        int bid, int tid, int nthr, const void* tmap, unsigned long long* bar, const int* done_flag)
{
    typedef B7<LOGM, LOGTC> P;
    constexpr int TC = P::TC, LOGTOP = LOGM - P::LOGR1;      // first middle stage: blocks of M / R1
    const int ntile = g.Lx / TC;
    const int x0 = (bid % ntile) * TC, zq = bid / ntile;
    const int kz = (int)brev((unsigned)zq, g.logpz);
    const int kzp = IS3D ? (kz <= g.nz ? kz : g.pz - kz) : 0;
    const T sz = (IS3D && kz > g.nz) ? (T)-1 : (T)1;
    const T* Kt = Kc + ((long)kzp * ntile + bid % ntile) * kc_tile_elems(g);
    constexpr int EW = (int)sizeof(cx<T>) / 8;
#if defined(__CUDA_ARCH__)
    if (tid == 0) {
        for (int c = 0; c < 3; c++) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((unsigned)__cvta_generic_to_shared(bar + c)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        for (int c = 0; c < 3; c++) {
            const unsigned b32 = (unsigned)__cvta_generic_to_shared(bar + c);
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b32), "r"(P::M * TC * (int)sizeof(cx<T>)) : "memory");
#pragma unroll
            for (int r0 = 0; r0 < P::M; r0 += P::RB) {
                const unsigned dst = (unsigned)__cvta_generic_to_shared(s + c * P::CS + r0 * TC);
                asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                             ::"r"(dst), "l"(tmap), "r"(x0 * EW), "r"(r0), "r"(zq), "r"(c), "r"(b32) : "memory");
            }
        }
        prefetch_l2_bulk(Kt, (unsigned)(kc_tile_elems(g) * sizeof(T)));
    }
    const int done = *reinterpret_cast<const volatile int*>(done_flag);
#else
    const int done = 0; (void)done_flag; (void)tmap; (void)EW;
    for (int c = 0; c < 3; c++)
        for (int j = 0; j < P::M; j++)
            for (int col = 0; col < TC; col++) s[c * P::CS + j * TC + col] = S[(long)c * g.comp + (long)zq * g.plane + (long)j * g.Lx + x0 + col];
#endif
    // twiddles of the first stage while the tile is in flight
    const twfl<T, P::R1> tf = b7_fl_tw<T, P::R1>(tw, logtw, LOGM + 1, (tid >> LOGTC) & (P::SUB1 - 1));
    MM_SYNC();      // the barrier words are initialised before anyone polls them
    b7_first<LOGM, LOGTC, NTHR, T>(s, tf, tw, logtw, tid, nthr, bar);
    if (done) return;      // every thread that owns an item has seen all three loads land
    kset<T, IS3D ? 48 : 32> kpre;
    b7_fwd_mids<LOGM, LOGTC, LOGTOP, IS3D, NTHR, T>(s, tw, logtw, Kt, tid, nthr, kpre);
    b7_mul8<LOGM, LOGTC, IS3D, NTHR, T>(s, kpre, Kt, sz, tid, nthr);
    b7_inv_mids<LOGM, LOGTC, 6, LOGTOP, NTHR, T>(s, tw, logtw, tid, nthr);
    const twfl<T, P::R1> tl = b7_fl_tw<T, P::R1>(tw, logtw, LOGM + 1, (tid >> LOGTC) & (P::SUB1 - 1));
    MM_SYNC();
    b7_last<LOGM, LOGTC, NTHR, T>(s, tl, tw, logtw, tid, nthr);
#if defined(__CUDA_ARCH__)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // the threads' tile writes before the async-proxy reads
    __syncthreads();
    if (tid == 0) {
        for (int c = 0; c < 3; c++)
#pragma unroll
            for (int r0 = 0; r0 < P::M; r0 += P::RB) {
                const unsigned src = (unsigned)__cvta_generic_to_shared(s + c * P::CS + r0 * TC);
                asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
                             ::"l"(tmap), "r"(x0 * EW), "r"(r0), "r"(zq), "r"(c), "r"(src) : "memory");
            }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");      // the tile must outlive the copies
    }
#else
    for (int c = 0; c < 3; c++)
        for (int j = 0; j < P::M; j++)
            for (int col = 0; col < TC; col++) S[(long)c * g.comp + (long)zq * g.plane + (long)j * g.Lx + x0 + col] = s[c * P::CS + j * TC + col];
#endif
}

}  // namespace mm
