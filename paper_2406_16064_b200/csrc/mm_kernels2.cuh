// mm_kernels2.cuh — v2 bodies of the convolution passes: same math and memory layout as
// mm_kernels.cuh (which stays as the fallback for tiny meshes), restructured for instruction
// count and shared-memory traffic:
//   * global loads / stores are fused into the first / last radix stage of each transform
//     (zero-padding and cropping included), so the tile makes 8 shared-memory round trips in
//     pass B instead of 16;
//   * in pass B the last forward stage, the spectral 3x3 multiply (Eq. 8 in k-space,
//     PAPER.md:138) and the first inverse stage run in registers on the three components of one
//     column;
//   * the z transform of passes A / C (nz <= 32) runs in registers, one thread per x position;
//   * all index arithmetic is shifts and masks; twiddle powers are shared by the three components
//     (pass B) or by a group of lines (passes A / C); pass B moves 16 bytes per shared-memory access.
#pragma once
#include "mm_fft.cuh"
#include "mm_kernels.cuh"

namespace mm {

// Pass B tile layouts.  Row-major (CM = false): element (row, comp, col) at row*3*TC + comp*TC + col — rows
// are loaded / stored by the threads with plain global accesses.  Component-major (CM = true):
// comp*py*TC + row*TC + col — each component's rows are dense, which is the box shape a TMA tensor-map
// copy deposits and picks up; used by the TMA form of the kernel.
template <bool CM> MM_HD int rsB(const Geom& g) { return CM ? g.TC : 3 * g.TC; }
template <bool CM> MM_HD int csB(const Geom& g) { return CM ? g.py * g.TC : g.TC; }

template <typename E, typename T> MM_HD E ldv(const cx<T>* p) { return *reinterpret_cast<const E*>(p); }
template <typename E, typename T> MM_HD void stv(cx<T>* p, const E& v) { *reinterpret_cast<E*>(p) = v; }

// ------------------------------------------------------------------------------------------------
// Pass B v2
// ------------------------------------------------------------------------------------------------
// first stage: load (global, or CM: the rows a TMA copy left in the first m rows of the tile) + zero-pad
// twiddle + radix R on both blocks
// spin until phase 0 of the shared-memory mbarrier has completed (a TMA load has landed); host: no-op
MM_HD void mbar_wait0(unsigned long long* bar)
{
#if defined(__CUDA_ARCH__)
    const unsigned b32 = (unsigned)__cvta_generic_to_shared(bar);
    unsigned done = 0;
    while (!done)
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }" : "=r"(done) : "r"(b32), "r"(0) : "memory");
#else
    (void)bar;
#endif
}

// `bars` (CM only, may be null): one mbarrier per component; the rows of component c are in the tile once
// bars[c] has completed, so the stage starts on component 0 while the other two are still in flight
template <typename T, int V, int R, bool CM>
MM_HD void yB_first(const Geom& g, const cx<T>* Sz, cx<T>* s, twiddles<T> tw, int tid, int nthr, unsigned long long* bars = nullptr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = rsB<CM>(g), cs = csB<CM>(g);
    const int m = g.ny, n = g.py, sub = m / R;
    for (int f = tid; f < sub * LC; f += nthr) {
        const int lc = f & (LC - 1), i = f >> logLC;
        cx<T> pw[R], wp[R];
        pad_twiddles<T, R>(tw.get(i, n), wp);
        if (R > 1 && i != 0) twiddle_powers<T, R>(cmul(wp[0], wp[0]), pw);      // w_m^i = (w_n^i)^2
        // fp64 (one column per item, 255-register kernel): the global loads of all three components are in
        // flight before the first butterfly; fp32 (128-register kernel) loads component by component —
        // preloading there costs registers and measured 1.5 % slower
        constexpr bool PRE = !CM && V == 1 && sizeof(T) == 8;
        constexpr int NA = PRE ? 3 : 1;
        E av[NA][R];
        const cx<T>* src0 = Sz + (long)i * g.Lx + lc * V;
        if (PRE) {
#pragma unroll
            for (int c = 0; c < 3; c++)
#pragma unroll
                for (int r = 0; r < R; r++) av[c % NA][r] = ldv<E, T>(src0 + (long)c * g.comp + (long)r * sub * g.Lx);
        }
#pragma unroll
        for (int c = 0; c < 3; c++) {
            cx<T>* dst = s + (i) * pitch + c * cs + lc * V;
            const int rs = (sub) * pitch, mo = (m) * pitch;
            E a[R], u[R];
            if (CM && bars != nullptr) mbar_wait0(bars + c);
#pragma unroll
            for (int r = 0; r < R; r++) a[r] = CM ? ldv<E, T>(dst + r * rs) : (PRE ? av[c % NA][r] : ldv<E, T>(src0 + (long)c * g.comp + (long)r * sub * g.Lx));
#pragma unroll
            for (int r = 0; r < R; r++) u[r] = cmul(a[r], wp[r]);
            rad<E, R>::fwd(a);
            rad<E, R>::fwd(u);
            if (i != 0) {
#pragma unroll
                for (int r = 1; r < R; r++) { a[r] = cmul(a[r], pw[r]); u[r] = cmul(u[r], pw[r]); }
            }
#pragma unroll
            for (int r = 0; r < R; r++) { stv<E, T>(dst + r * rs, a[r]); stv<E, T>(dst + mo + r * rs, u[r]); }
        }
    }
}

// last stage: inverse radix R on both blocks + crop combine + store (global, or CM: in place in the tile)
template <typename T, int V, int R, bool CM>
MM_HD void yB_last(const Geom& g, cx<T>* Sz, cx<T>* s, twiddles<T> tw, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = rsB<CM>(g), cs = csB<CM>(g);
    const int m = g.ny, n = g.py, sub = m / R;
    for (int f = tid; f < sub * LC; f += nthr) {
        const int lc = f & (LC - 1), i = f >> logLC;
        cx<T> pw[R], wp[R];
        pad_twiddles<T, R>(tw.get(i, n), wp);
        if (R > 1 && i != 0) twiddle_powers<T, R>(cmul(wp[0], wp[0]), pw);
#pragma unroll
        for (int c = 0; c < 3; c++) {
            cx<T>* dstg = Sz + (long)c * g.comp + (long)i * g.Lx + lc * V;
            cx<T>* src = s + (i) * pitch + c * cs + lc * V;
            const int rs = (sub) * pitch, mo = (m) * pitch;
            E a[R], u[R];
#pragma unroll
            for (int r = 0; r < R; r++) { a[r] = ldv<E, T>(src + r * rs); u[r] = ldv<E, T>(src + mo + r * rs); }
            if (i != 0) {
#pragma unroll
                for (int r = 1; r < R; r++) { a[r] = cmulc(a[r], pw[r]); u[r] = cmulc(u[r], pw[r]); }
            }
            rad<E, R>::inv(a);
            rad<E, R>::inv(u);
#pragma unroll
            for (int r = 0; r < R; r++) {
                const E o = a[r] + cmulc(u[r], wp[r]);
                if (CM) stv<E, T>(src + r * rs, o);      // back into the first m rows: a TMA copy stores them
                else stv<E, T>(dstg + (long)r * sub * g.Lx, o);
            }
        }
    }
}

// middle radix-8 stage (DIR = 0 forward DIF, 1 inverse DIT) on blocks of length Lc over all n points
template <typename T, int V, int DIR, bool CM>
MM_HD void yB_mid8(const Geom& g, cx<T>* s, int Lc, twiddles<T> tw, int tid, int nthr)
{
    typedef cvec<T, V> E;
    const int TC = g.TC, LC = TC / V, logLC = ilog2(LC), pitch = rsB<CM>(g), cs = csB<CM>(g);
    const int n = g.py, sub = Lc >> 3, logsub = ilog2(sub);
    for (int f = tid; f < (n >> 3) * LC; f += nthr) {
        const int lc = f & (LC - 1), b = f >> logLC;
        const int blk = b >> logsub, i = b & (sub - 1);
        cx<T> pw[8];
        if (i != 0) twiddle_powers<T, 8>(tw.get(i, Lc), pw);
        cx<T>* base = s + (blk * Lc + i) * pitch + lc * V;
        const int rs = (sub) * pitch;
#pragma unroll
        for (int c = 0; c < 3; c++) {
            cx<T>* p = base + c * cs;
            E v[8];
#pragma unroll
            for (int r = 0; r < 8; r++) v[r] = ldv<E, T>(p + r * rs);
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
            for (int r = 0; r < 8; r++) stv<E, T>(p + r * rs, v[r]);
        }
    }
}

template <typename T> struct alignas(16) kvec { T e[16 / sizeof(T)]; };

MM_HD void prefetch_l2_bulk(const void* p, unsigned bytes)
{
#if defined(__CUDA_ARCH__)
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
#else
    (void)p; (void)bytes;
#endif
}

// last forward radix-8 stage (Lc = 8) + multiply by K^ + first inverse stage, three components in
// registers.  An item is a column and a PAIR of 8-row blocks whose frequencies mirror each other (ky <-> py - ky,
// see kc_fill): t = 1 .. nbk/2 - 1 owns the blocks beta = t and nbk - t and reads ONE set of K^ (NJ/EPL 16-byte
// loads) for both — the second block uses it with the rows reversed and the odd components (xy, yz) negated;
// t = 0 owns the two self-mirrored blocks beta = 0 and nbk/2 and reads a set for each.  Kt = this CTA's tile of Kc.
template <typename T, bool IS3D, bool CM>
MM_HD void yB_mul8(const Geom& g, cx<T>* s, const T* Kt, T sz, int tid, int nthr)
{
    constexpr int NQ = IS3D ? 6 : 4, NJ = 8 * NQ, EPL = 16 / (int)sizeof(T), NJQ = NJ / EPL;
    const int TC = g.TC, logTC = ilog2(TC), pitch = rsB<CM>(g), cs = csB<CM>(g);
    const int nbk = g.py >> 3, lognbk = g.logpy - 3;
    for (int f = tid; f < (nbk >> 1) * TC; f += nthr) {
        const int col = f & (TC - 1), t = f >> logTC;
        // Rows of an 8-point block are taken cyclically rotated by t & 7: register slot r holds row
        // (r + t) & 7.  DFT_8 -> per-frequency real multiply -> IDFT_8 commutes with a cyclic shift (the
        // phase factors w8^(-g k) cancel), so the result lands in the right rows, and the lanes of a warp
        // (block offsets = 0 mod 256 bytes) hit different bank windows.
        int ro[8];
#pragma unroll
        for (int r = 0; r < 8; r++) ro[r] = ((r + t) & 7) * pitch;
        T K[NJ];
        {
            const T* Kp = Kt + (long)t * (NJ * TC) + col * EPL;
#pragma unroll
            for (int jq = 0; jq < NJQ; jq++) {
                const kvec<T> v = *reinterpret_cast<const kvec<T>*>(Kp + jq * TC * EPL);
#pragma unroll
                for (int e = 0; e < EPL; e++) K[jq * EPL + e] = v.e[e];
            }
        }
#pragma unroll
        for (int h = 0; h < 2; h++) {
            const int beta = h == 0 ? t : (t == 0 ? (nbk >> 1) : nbk - t);
            if (h == 1 && t == 0) {      // the second self-mirrored block has its own set (stored row-reversed and signed like a mirror)
                const T* Kp = Kt + (long)(nbk >> 1) * (NJ * TC) + col * EPL;
#pragma unroll
                for (int jq = 0; jq < NJQ; jq++) {
                    const kvec<T> v = *reinterpret_cast<const kvec<T>*>(Kp + jq * TC * EPL);
#pragma unroll
                    for (int e = 0; e < EPL; e++) K[jq * EPL + e] = v.e[e];
                }
            }
            cx<T>* p = s + ((int)brev((unsigned)beta, lognbk) * 8) * pitch + col;
            cx<T> M[3][8];
#pragma unroll
            for (int c = 0; c < 3; c++) {
#pragma unroll
                for (int r = 0; r < 8; r++) M[c][r] = p[ro[r] + c * cs];
                rad<cx<T>, 8>::fwd(M[c]);
            }
#pragma unroll
            for (int r = 0; r < 8; r++) {
                // second block: K_B[r][q] = +-K_A[7 - r][q] (odd components xy, yz change sign)
                const int kr = (h == 0 ? r : 7 - r) * NQ;
                const T so = h == 0 ? (T)1 : (T)-1;
                const T kxx = K[kr], kyy = K[kr + 1], kzz = K[kr + 2], kxy = so * K[kr + 3];
                const cx<T> Mx = M[0][r], My = M[1][r], Mz = M[2][r];
                if (IS3D) {
                    const T kxz = sz * K[kr + (IS3D ? 4 : 0)], kyz = (so * sz) * K[kr + (IS3D ? 5 : 0)];
                    M[0][r] = lin3<T>(Mx, kxx, My, kxy, Mz, kxz);
                    M[1][r] = lin3<T>(Mx, kxy, My, kyy, Mz, kyz);
                    M[2][r] = lin3<T>(Mx, kxz, My, kyz, Mz, kzz);
                } else {
                    M[0][r] = lin2<T>(Mx, kxx, My, kxy);
                    M[1][r] = lin2<T>(Mx, kxy, My, kyy);
                    M[2][r] = scale<T>(Mz, kzz);
                }
            }
#pragma unroll
            for (int c = 0; c < 3; c++) {
                rad<cx<T>, 8>::inv(M[c]);
#pragma unroll
                for (int r = 0; r < 8; r++) p[ro[r] + c * cs] = M[c][r];
            }
        }
    }
}

// stages of one tile; CM = false: first / last stage move the rows from / to Sz themselves
// returns false when `done` (the step controller's flag, read by the caller; tested only after the first stage so
// that the load is off the critical path) stops the pass early
template <typename T, int V, bool CM>
MM_HD bool y_conv_stages(const Geom& g, cx<T>* Sz, const T* Kt, T sz, twiddles<T> tw, cx<T>* s, int tid, int nthr, unsigned long long* bars = nullptr,
                         int done = 0)
{
    const int m = g.ny;
    const bool is3d = g.nz > 1;
    const int R1 = first_radix(m);
    // first / last stage: one column per item when column pairs would leave threads without an item
    const bool narrow = V > 1 && (m / R1) * (g.TC / V) < nthr;
    if (narrow) {
        if (R1 == 8) yB_first<T, 1, 8, CM>(g, Sz, s, tw, tid, nthr, bars);
        else if (R1 == 4) yB_first<T, 1, 4, CM>(g, Sz, s, tw, tid, nthr, bars);
        else yB_first<T, 1, 2, CM>(g, Sz, s, tw, tid, nthr, bars);
    } else if (R1 == 8) yB_first<T, V, 8, CM>(g, Sz, s, tw, tid, nthr, bars);
    else if (R1 == 4) yB_first<T, V, 4, CM>(g, Sz, s, tw, tid, nthr, bars);
    else yB_first<T, V, 2, CM>(g, Sz, s, tw, tid, nthr, bars);
    if (done) return false;
    MM_SYNC();
    // the K^ tile of the multiply stage towards L2 while the middle stages run
    if (!CM && !(g.flags & 1) && tid == 0) prefetch_l2_bulk(Kt, (unsigned)(kc_tile_elems(g) * sizeof(T)));
    int Lc = m / R1;
    for (; Lc > 8; Lc >>= 3) { yB_mid8<T, V, 0, CM>(g, s, Lc, tw, tid, nthr); MM_SYNC(); }
    if (is3d) yB_mul8<T, true, CM>(g, s, Kt, sz, tid, nthr);
    else yB_mul8<T, false, CM>(g, s, Kt, sz, tid, nthr);
    MM_SYNC();
    for (Lc = 64; Lc <= m / R1; Lc <<= 3) { yB_mid8<T, V, 1, CM>(g, s, Lc, tw, tid, nthr); MM_SYNC(); }
    if (narrow) {
        if (R1 == 8) yB_last<T, 1, 8, CM>(g, Sz, s, tw, tid, nthr);
        else if (R1 == 4) yB_last<T, 1, 4, CM>(g, Sz, s, tw, tid, nthr);
        else yB_last<T, 1, 2, CM>(g, Sz, s, tw, tid, nthr);
    } else if (R1 == 8) yB_last<T, V, 8, CM>(g, Sz, s, tw, tid, nthr);
    else if (R1 == 4) yB_last<T, V, 4, CM>(g, Sz, s, tw, tid, nthr);
    else yB_last<T, V, 2, CM>(g, Sz, s, tw, tid, nthr);
    return true;
}

// requires ny >= 16 (so the schedule has >= 2 stages and ends with radix 8) and TC % V == 0
template <typename T, int V>
MM_HD void y_conv_body2(const Geom g, cx<T>* __restrict__ S, const T* __restrict__ Kc, twiddles<T> tw, cx<T>* s,
                        int bid, int tid, int nthr)
{
    const int ntile = g.Lx / g.TC;
    const int x0 = (bid % ntile) * g.TC, zq = bid / ntile;
    const int kz = (int)brev((unsigned)zq, g.logpz);
    const bool is3d = g.nz > 1;
    const int kzp = is3d ? (kz <= g.nz ? kz : g.pz - kz) : 0;
    const T sz = (is3d && kz > g.nz) ? (T)-1 : (T)1;
    const T* Kt = Kc + ((long)kzp * ntile + bid % ntile) * kc_tile_elems(g);
    y_conv_stages<T, V, false>(g, S + (long)zq * g.plane + x0, Kt, sz, tw, s, tid, nthr);
}

// TMA form: the rows of the tile travel as tensor-map box copies (cp.async.bulk.tensor, boxes of TC columns x
// <= 256 rows of one component) between S and the component-major tile; no thread issues a global load or
// store of S.  `tmap` = CUtensorMap of S as (x, j, zpos, comp) in 8-byte (fp32) / 2 x 8-byte (fp64) elements,
// `bar` = an 8-byte shared-memory mbarrier.  On the host (emulation) the copies are plain loops.
template <typename T, int V>
MM_HD void y_conv_body5(const Geom g, cx<T>* __restrict__ S, const T* __restrict__ Kc, twiddles<T> tw, cx<T>* s,
                        int bid, int tid, int nthr, const void* tmap, unsigned long long* bar, const int* done_flag = nullptr)
{
    const int ntile = g.Lx / g.TC;
    const int x0 = (bid % ntile) * g.TC, zq = bid / ntile;
    const int kz = (int)brev((unsigned)zq, g.logpz);
    const bool is3d = g.nz > 1;
    const int kzp = is3d ? (kz <= g.nz ? kz : g.pz - kz) : 0;
    const T sz = (is3d && kz > g.nz) ? (T)-1 : (T)1;
    const T* Kt = Kc + ((long)kzp * ntile + bid % ntile) * kc_tile_elems(g);
    const int RB = g.ny < 256 ? g.ny : 256, cs = csB<true>(g);
    constexpr int EW = (int)sizeof(cx<T>) / 8;      // 8-byte tensor-map elements per complex number
#if defined(__CUDA_ARCH__)
    // one mbarrier per component (bar[0..2]); the loads are issued before the step controller's `done` flag
    // has arrived (a kernel enqueued after the stop condition loads its tile for nothing and returns)
    if (tid == 0) {
        for (int c = 0; c < 3; c++) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"((unsigned)__cvta_generic_to_shared(bar + c)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        for (int c = 0; c < 3; c++) {
            const unsigned b32 = (unsigned)__cvta_generic_to_shared(bar + c);
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b32), "r"(g.ny * g.TC * (int)sizeof(cx<T>)) : "memory");
            for (int r0 = 0; r0 < g.ny; r0 += RB) {
                const unsigned dst = (unsigned)__cvta_generic_to_shared(s + c * cs + r0 * g.TC);
                asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                             ::"r"(dst), "l"(tmap), "r"(x0 * EW), "r"(r0), "r"(zq), "r"(c), "r"(b32) : "memory");
            }
        }
        // the K^ tile of the multiply stage follows the rows towards L2
        if (!(g.flags & 1)) prefetch_l2_bulk(Kt, (unsigned)(kc_tile_elems(g) * sizeof(T)));
    }
    const int done = done_flag ? *reinterpret_cast<const volatile int*>(done_flag) : 0;
    __syncthreads();      // the barrier words are initialised before anyone polls them
#else
    const int done = 0; (void)done_flag;
    (void)tmap; (void)bar; (void)RB; (void)EW;
    for (int c = 0; c < 3; c++)
        for (int j = 0; j < g.ny; j++)
            for (int col = 0; col < g.TC; col++) s[c * cs + j * g.TC + col] = S[(long)c * g.comp + (long)zq * g.plane + (long)j * g.Lx + x0 + col];
#endif
    if (!y_conv_stages<T, V, true>(g, (cx<T>*)nullptr, Kt, sz, tw, s, tid, nthr, bar, done)) return;      // every thread has seen all three loads land
#if defined(__CUDA_ARCH__)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // the threads' tile writes before the async-proxy reads
    __syncthreads();
    if (tid == 0) {
        for (int c = 0; c < 3; c++)
            for (int r0 = 0; r0 < g.ny; r0 += RB) {
                const unsigned src = (unsigned)__cvta_generic_to_shared(s + c * cs + r0 * g.TC);
                asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];"
                             ::"l"(tmap), "r"(x0 * EW), "r"(r0), "r"(zq), "r"(c), "r"(src) : "memory");
            }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");      // the tile must outlive the copies
    }
#else
    for (int c = 0; c < 3; c++)
        for (int j = 0; j < g.ny; j++)
            for (int col = 0; col < g.TC; col++) S[(long)c * g.comp + (long)zq * g.plane + (long)j * g.Lx + x0 + col] = s[c * cs + j * g.TC + col];
#endif
}

// ------------------------------------------------------------------------------------------------
// Passes A / C v2 (x transform of packed pairs with m = nx/2, n = nx; z transform in registers)
// ------------------------------------------------------------------------------------------------
// first x stage: load Ms*m pairs from global (i fastest: coalesced), pad twiddle, radix R, both blocks.
// A thread keeps one i (butterfly index) and walks the lines: the pad twiddles w_n^(i + r sub) and the
// stage twiddles are loaded / formed once per thread, not once per line.
template <typename T, int R, bool PAD>
MM_HD void xA_first(const Geom& g, const T* mc, const T* Ms, cx<T>* s, int pitch, int j0, twiddles<T> tw, int tid, int nthr)
{
    const int n = g.nx, m = n / 2, sub = m / R, L = g.G * g.nz, lognz = ilog2(g.nz);
    const int isub = sub < nthr ? sub : nthr, logisub = ilog2(isub), lstep = nthr >> logisub;
    for (int i = tid & (isub - 1); i < sub; i += isub) {
        cx<T> wp[R], pw[R];
#pragma unroll
        for (int r = 0; r < R; r++) wp[r] = tw.get(i + r * sub, n);
        if (R > 1 && i != 0) twiddle_powers<T, R>(tw.get(i, m), pw);
        // fp64: two lines per trip, the global loads of both in flight before the first butterfly (the load latency is
        // exposed once per trip: 29 % of the pass's stall samples; cfg4 pass A 188.8 -> 178.7 us).  fp32 keeps one line:
        // two need more than the 85 registers of three CTAs per SM (measured 78.8 -> 87.0 us with two).
        constexpr int NB = sizeof(T) == 8 ? 2 : 1;
        for (int l0 = tid >> logisub; l0 < L; l0 += NB * lstep) {
            cx<T> a[NB][R], u[NB][R];
            cx<T> mm2[NB][R], ms2[NB][R];
#pragma unroll
            for (int b = 0; b < NB; b++) {
                const int l = l0 + b * lstep;
                if (l < L) {
                    const int gg = l >> lognz, z = l & (g.nz - 1);
                    const long row = ((long)z * g.ny + (j0 + gg)) * g.nx + 2 * i;
#pragma unroll
                    for (int r = 0; r < R; r++) {
                        mm2[b][r] = *reinterpret_cast<const cx<T>*>(mc + row + 2 * r * sub);
                        ms2[b][r] = *reinterpret_cast<const cx<T>*>(Ms + row + 2 * r * sub);
                    }
                }
            }
#pragma unroll
            for (int b = 0; b < NB; b++) {
                const int l = l0 + b * lstep;
                if (l < L) {
#pragma unroll
                    for (int r = 0; r < R; r++) {
                        a[b][r] = mk<T>(ms2[b][r].x == (T)0 ? (T)0 : ms2[b][r].x * mm2[b][r].x, ms2[b][r].y == (T)0 ? (T)0 : ms2[b][r].y * mm2[b][r].y);
                        u[b][r] = cmul(a[b][r], wp[r]);
                    }
                    rad<cx<T>, R>::fwd(a[b]);
                    rad<cx<T>, R>::fwd(u[b]);
                    if (R > 1 && i != 0) {
#pragma unroll
                        for (int r = 1; r < R; r++) { a[b][r] = cmul(a[b][r], pw[r]); u[b][r] = cmul(u[b][r], pw[r]); }
                    }
                    cx<T>* dst = s + ppos(i, PAD) * pitch + l;
                    const int sp = ppos(sub, PAD) * pitch, mp = ppos(m, PAD) * pitch;
#pragma unroll
                    for (int r = 0; r < R; r++) { dst[r * sp] = a[b][r]; dst[mp + r * sp] = u[b][r]; }
                }
            }
        }
    }
}

// last x stage of pass C: inverse radix R on both blocks, crop combine, scale, store H_d pairs (same
// thread -> (i, lines) mapping as xA_first)
template <typename T, int R, bool PAD>
MM_HD void xC_last(const Geom& g, T* Hc, const cx<T>* s, int pitch, int j0, T inv_scale, twiddles<T> tw, int tid, int nthr)
{
    const int n = g.nx, m = n / 2, sub = m / R, L = g.G * g.nz, lognz = ilog2(g.nz);
    const int isub = sub < nthr ? sub : nthr, logisub = ilog2(isub), lstep = nthr >> logisub;
    for (int i = tid & (isub - 1); i < sub; i += isub) {
        cx<T> wp[R], pw[R];
#pragma unroll
        for (int r = 0; r < R; r++) wp[r] = scale(tw.get(i + r * sub, n), inv_scale);      // 1/P folded into the crop twiddle
        if (R > 1 && i != 0) twiddle_powers<T, R>(tw.get(i, m), pw);
        for (int l = tid >> logisub; l < L; l += lstep) {
            const int gg = l >> lognz, z = l & (g.nz - 1);
            T* hrow = Hc + ((long)z * g.ny + (j0 + gg)) * g.nx + 2 * i;
            const cx<T>* src = s + ppos(i, PAD) * pitch + l;
            const int sp = ppos(sub, PAD) * pitch, mp = ppos(m, PAD) * pitch;
            cx<T> a[R], u[R];
#pragma unroll
            for (int r = 0; r < R; r++) { a[r] = src[r * sp]; u[r] = src[mp + r * sp]; }
            if (R > 1 && i != 0) {
#pragma unroll
                for (int r = 1; r < R; r++) { a[r] = cmulc(a[r], pw[r]); u[r] = cmulc(u[r], pw[r]); }
            }
            rad<cx<T>, R>::inv(a);
            rad<cx<T>, R>::inv(u);
#pragma unroll
            for (int r = 0; r < R; r++)
                *reinterpret_cast<cx<T>*>(hrow + 2 * r * sub) = scale(a[r], inv_scale) + cmulc(u[r], wp[r]);
        }
    }
}

// z transform in registers, inverse + crop: S -> tile
template <typename T, int NZ, bool PAD>
MM_HD void zC_regs(const Geom& g, const cx<T>* Sc, cx<T>* s, int pitch, int j0, twiddles<T> tw, int tid, int nthr)
{
    const int np = g.nx + 1;
    for (int f = tid; f < np * g.G; f += nthr) {
        const int xp = f % np, gg = f / np;
        cx<T>* dst = s + ppos(xp, PAD) * pitch + gg * NZ;
        const cx<T>* src = Sc + (long)(j0 + gg) * g.Lx + xp;
        cx<T> a[NZ], u[NZ];
#pragma unroll
        for (int z = 0; z < NZ; z++) { a[z] = src[(long)z * g.plane]; u[z] = src[(long)(NZ + z) * g.plane]; }
        rad<cx<T>, NZ>::inv(a);
        rad<cx<T>, NZ>::inv(u);
        dst[0] = a[0] + u[0];
#pragma unroll
        for (int z = 1; z < NZ; z++) dst[z] = a[z] + rot_wc<T, 2 * NZ>(u[z], z);      // conj(w_2NZ^z), an immediate
    }
}

}  // namespace mm
