// mm_lib.cu — libmm.so: the C ABI of include/mm.h, its host runtime and the __global__ kernels.
// Hand-written CUDA for sm_100a; no cuFFT, no cuBLAS, no CPU fallback.
#include <cuda.h>
#include <cuda_runtime.h>
#include <cooperative_groups.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <string>
#include <vector>

#include "../../include/mm.h"
#include "mm_fft.cuh"
#include "mm_kernels.cuh"
#include "mm_kernels2.cuh"
#include "mm_passAC.cuh"
#include "mm_passB7.cuh"
#include "mm_passB3.cuh"
#include "mm_passB4.cuh"
#include "mm_llg.cuh"

#ifndef MM_OCC_A
#define MM_OCC_A 3      // resident CTAs per SM the fp32 pass A kernel is compiled for
#endif
#ifndef MM_B5_THR
#define MM_B5_THR 512
#define MM_B5_OCC 1
#endif
#ifndef MM_OCC_C
#define MM_OCC_C 2
#endif

extern "C" void mm_newell_near_box(int bx, int by, int bz, double dx, double dy, double dz, double* out);

namespace mm {

static const double MU0 = 4.0e-7 * 3.14159265358979323846264338327950288;
static const int ALL_TERMS = 63;      // LocalP::terms: exchange | DMI | uniaxial | Zeeman | demag | cubic

// Device-resident step controller state.
struct DevState {
    double dt, t, tol, err, maxk, t_end, stop_dmdt;
    unsigned long long err_bits, maxk_bits;
    int accepted, done, nan, mode;     // mode: 0 single step, 1 relax, 2 run_until
    long long nacc, nrej, nsteps;
    unsigned long long th_step;        // thermal field: step attempts since mm_set_temperature (Philox counter word)
    long long nrhs;                    // RHS evaluations of all step attempts; with nacc / nrej: totals since mm_set_workspace (mm_get_stats)
};

// ------------------------------------------------------------------------------------------------
// __global__ wrappers of the convolution passes
// ------------------------------------------------------------------------------------------------
extern __shared__ __align__(128) unsigned char mm_smem[];

template <typename T>
__global__ void __launch_bounds__(256) fwd_xz_kernel(Geom g, const T* m, const T* Ms, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    if (st->done) return;
    fwd_xz_body<T>(g, m, Ms, S, tw, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, blockDim.x);
}
template <typename T>
__global__ void __launch_bounds__(512) y_conv_kernel(Geom g, cx<T>* S, const T* Kh, twiddles<T> tw, const DevState* st)
{
    if (st->done) return;
    y_conv_body<T>(g, S, Kh, tw, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, blockDim.x);
}
template <typename T>
__global__ void __launch_bounds__(256) inv_zx_kernel(Geom g, const cx<T>* S, T* Hd, twiddles<T> tw, T inv_scale, const DevState* st)
{
    if (st->done) return;
    inv_zx_body<T>(g, S, Hd, tw, inv_scale, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, blockDim.x);
}

// v2 wrappers (mm_kernels2.cuh)
template <typename T, int NZ, bool PAD>
__global__ void __launch_bounds__(256, sizeof(T) == 8 ? 1 : MM_OCC_A) fwd_xz2_kernel(Geom g, const T* m, const T* Ms, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    if (st->done) return;
    fwd_xz_body3<T, NZ, PAD>(g, m, Ms, S, tw, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, blockDim.x);
}
template <typename T, int V>
__global__ void __launch_bounds__(sizeof(T) == 8 ? 256 : 512) y_conv2_kernel(Geom g, cx<T>* S, const T* Kh, twiddles<T> tw, const DevState* st)
{
    if (st->done) return;
    y_conv_body2<T, V>(g, S, Kh, tw, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, blockDim.x);
}
// TMA form of pass B: tile rows move as tensor-map box copies (y_conv_body5)
template <typename T, int V>
__global__ void __launch_bounds__(MM_B5_THR, MM_B5_OCC) y_conv5_kernel(Geom g, cx<T>* S, const T* Kh, twiddles<T> tw, const DevState* st,
                                                                             const __grid_constant__ CUtensorMap tmS)
{
    __shared__ __align__(8) unsigned long long bar[3];
    y_conv_body5<T, V>(g, S, Kh, tw, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, blockDim.x, &tmS, bar, &st->done);
}
// half-tile form (mm_passB3.cuh): the long-line path; reads S, writes the second spectrum buffer S2
template <typename T, int V>
__global__ void __launch_bounds__(256) y_conv3_kernel(Geom g, const cx<T>* S, cx<T>* S2, const T* Kh, twiddles<T> tw, const DevState* st)
{
    if (st->done) return;
    y_conv_body3<T, V>(g, S, S2, Kh, tw, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, blockDim.x);
}
// cluster form (mm_passB4.cuh): the long-line path; Q CTAs of a thread-block cluster share one line through
// distributed shared memory
template <typename T, int V, int Q>
__global__ void __launch_bounds__(256, sizeof(T) == 8 ? 1 : 2) y_conv4_kernel(Geom g, cx<T>* S, const T* Kh, twiddles<T> tw, const DevState* st)
{
    if (st->done) return;      // the same for every CTA of the cluster
    namespace cg = cooperative_groups;
    cg::cluster_group cl = cg::this_cluster();
    const int q = (int)cl.block_rank(), tile = (int)(blockIdx.x / Q);
    cx<T>* s = reinterpret_cast<cx<T>*>(mm_smem);
    y_conv_body4_compute<T, V, Q>(g, S, Kh, tw, s, tile, q, threadIdx.x, blockDim.x);
    cl.sync();      // every block's z_q is complete and visible across the cluster
    cx<T>* tiles[Q];
#pragma unroll
    for (int qq = 0; qq < Q; qq++) tiles[qq] = cl.map_shared_rank(s, qq);
    y_conv_body4_combine<T, V, Q>(g, S, tiles, tile, q, threadIdx.x, blockDim.x);
    cl.sync();      // nobody leaves while a neighbour still reads its tile
}
// compile-time specialised form of the TMA pass B (mm_passB7.cuh): ny = 2^LOGM; fp32: TC = 4, 256 threads; fp64: TC = 2,
// 128 threads (rows of 32 bytes and tiles of py * 96 bytes in both; two CTAs per SM)
// ny = 1024: one CTA per SM with twice the threads (tile py * 96 bytes = 196 KB)
// NARROW (fp32, ny = 512 / 1024): tiles of 2 columns (16-byte rows, 48 / 96 KB), 128 / 256 threads, four / two CTAs per
// SM — the phases of more, smaller CTAs interleave better (cfg4 pass B 186.5 -> 182 us, film 1024^2 45.3 -> 43.0 us,
// profiles/r02_experiments.md)
template <typename T, int LOGM, bool IS3D, bool NARROW = false>
__global__ void __launch_bounds__((NARROW || sizeof(T) == 8 ? 128 : 256) * (LOGM >= 10 ? 2 : 1), (NARROW ? 4 : 2) / (LOGM >= 10 ? 2 : 1)) y_conv7_kernel(Geom g, cx<T>* S, const T* Kc, twiddles<T> tw, int logtw, const DevState* st,
                                                                                const __grid_constant__ CUtensorMap tmS)
{
    __shared__ __align__(8) unsigned long long bar[3];
    constexpr int LOGTC = (NARROW || sizeof(T) == 8) ? 1 : 2, NTHR = (NARROW || sizeof(T) == 8 ? 128 : 256) * (LOGM >= 10 ? 2 : 1);
    y_conv_body7<LOGM, LOGTC, IS3D, NTHR, T>(g, S, Kc, tw, logtw, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, NTHR, &tmS, bar, &st->done);
}
template <typename T, int NZ, bool PAD>
__global__ void __launch_bounds__(256, sizeof(T) == 8 ? 1 : MM_OCC_C) inv_zx2_kernel(Geom g, const cx<T>* S, T* Hd, twiddles<T> tw, T inv_scale, const DevState* st)
{
    if (st->done) return;
    inv_zx_body3<T, NZ, PAD>(g, S, Hd, tw, inv_scale, reinterpret_cast<cx<T>*>(mm_smem), blockIdx.x, threadIdx.x, blockDim.x);
}

// ------------------------------------------------------------------------------------------------
// Fused local field + LL torque + RK stage + reductions
// ------------------------------------------------------------------------------------------------
template <typename T> struct StageArgs {
    const T* m0;          // step start magnetisation
    const T* kprev[6];    // earlier stage derivatives k_0..k_{s-1}
    T* ynext;             // next stage input (or the RK4 solution); may be NULL
    T coef[7];            // ynext = m0 + dt * sum_{j<=s} coef[j] k_j
    T ecoef[7];           // E = dt * sum_{j<=s} ecoef[j] k_j   (do_err)
    T cstage;             // stage time = t + cstage * dt (time-dependent current)
    T wcoef[7];           // Cayley (MODE 2): omega of THIS stage = dt * sum_{j<s} wcoef[j] k_j, k_j = d omega/dt of stage j
    int s;                // index of this stage
    int do_err, do_maxk;
};

__device__ __forceinline__ unsigned long long norm_bits(float v) { return (unsigned long long)__float_as_uint(v); }
__device__ __forceinline__ unsigned long long norm_bits(double v) { return (unsigned long long)__double_as_longlong(v); }

__device__ __forceinline__ void block_max_bits(unsigned long long v, unsigned long long* dst)
{
    // non-negative IEEE values order like their bit patterns; a NaN pattern beats everything
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
        v = w > v ? w : v;
    }
    __shared__ unsigned long long red[32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) red[wid] = v;
    __syncthreads();
    if (wid == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        v = lane < nw ? red[lane] : 0ull;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
            v = w > v ? w : v;
        }
        if (lane == 0 && v != 0ull) atomicMax(dst, v);
    }
    __syncthreads();
}

// Warp-level form of block_max_bits for the vectorised stage kernel: no shared memory, no block barrier; a
// warp touches the global word only when it can raise it (the plain read may be stale, which only costs
// a redundant atomicMax).
__device__ __forceinline__ void warp_max_bits(unsigned long long v, unsigned long long* dst)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
        v = w > v ? w : v;
    }
    if ((threadIdx.x & 31) == 0 && v != 0ull && v > *reinterpret_cast<volatile unsigned long long*>(dst)) atomicMax(dst, v);
}

// From the total field h of a cell (every H_eff term, plus the thermal field during a step) to the stage's output:
// MODE 0 the field itself; MODE 1 dm/dt = Eq. 37 with the Slonczewski terms folded into the field (Eq. 40,
// PAPER.md:319) plus f_stt x m; MODE 2 d omega/dt of Eq. 49 at omega = w with f of Eq. 44.
// *kn = |dm/dt| when want_kn (MODE 2; MODE 1 takes it from the result).
template <typename T, int MODE>
__device__ __forceinline__ v3<T> stage_result(const LocalP<T>& lp, v3<T> mi, v3<T> h, v3<T> tau, v3<T> w, bool want_kn, T* kn)
{
    if (MODE == 0) return h;
    if (lp.sl_on) h = add_slonczewski<T>(lp, mi, h);
    if (MODE == 1) {
        v3<T> r = ll_torque<T>(lp, mi, h);
        if (lp.stt_on) { const v3<T> c = cross<T>(stt_f<T>(lp, mi, tau), mi); r.x += c.x; r.y += c.y; r.z += c.z; }
        return r;
    }
    v3<T> f = llg_f<T>(lp, mi, h);
    if (lp.stt_on) { const v3<T> fs = stt_f<T>(lp, mi, tau); f.x += fs.x; f.y += fs.y; f.z += fs.z; }
    if (want_kn) { const v3<T> c = cross<T>(f, mi); *kn = sqrt(c.x * c.x + c.y * c.y + c.z * c.z); }
    return cayley_domega<T>(w, f);
}

// u(t) / u of the Zhang-Li current at this stage's time (1 when the current is constant)
template <typename T> __device__ __forceinline__ T stt_pulse(const LocalP<T>& lp, const DevState* st, T cstage)
{
    if (!lp.stt_on || (lp.stt_b == 0.0 && lp.stt_w == 0.0)) return (T)1;
    const double ts = st->t + (double)cstage * st->dt;
    return (T)(exp(-lp.stt_b * ts) * cos(lp.stt_w * ts));
}

// MODE 0: out = H_eff ; MODE 1: out = k = LL torque ; MODE 2: out = d omega/dt (Cayley form, Eq. 49); then the RK
// stage algebra selected at compile time: S earlier stages, NEXT (write the next stage input: m0 + dt sum a k, or
// Q(dt sum a k) m0 in MODE 2), ERR (embedded error norm), MAXK (max |dm/dt|).
// One thread per cell; indices by shifts (all mesh sizes are powers of two).
template <typename T, int MODE, int S, bool NEXT, bool ERR, bool MAXK>
__global__ void __launch_bounds__(256) llg_stage_kernel(Geom g, LocalP<T> lp, const T* __restrict__ y, const T* __restrict__ Ms,
                                                        const T* __restrict__ Hd, T* __restrict__ out, StageArgs<T> sa, DevState* st)
{
    if (st->done) return;
    const long N = g.N;
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    T errn = 0, kn = 0;
    if (q < N) {
        const T Msi = Ms[q];
        const bool live = Msi != (T)0;
        const int i = q & (g.nx - 1), j = (q >> g.lognx) & (g.ny - 1), k = q >> (g.lognx + g.logny);
        const v3<T> mi = ld3(y, N, q);
        v3<T> H = { 0, 0, 0 };
        if (Hd != nullptr) H = ld3(Hd, N, q);
        v3<T> kj[S > 0 ? S : 1];
#pragma unroll
        for (int jj = 0; jj < S; jj++) kj[jj] = ld3(sa.kprev[jj], N, q);
        v3<T> m0 = { 0, 0, 0 };
        if (NEXT) m0 = ld3(sa.m0, N, q);
        v3<T> tau = { 0, 0, 0 };
        H = local_field<T>(g, lp, y, Ms, i, j, k, q, live ? Msi : (T)1, mi, H, MODE == 0 ? nullptr : &tau);
        if (MODE >= 1) { const T fp = stt_pulse<T>(lp, st, sa.cstage); tau.x *= fp; tau.y *= fp; tau.z *= fp; }
        v3<T> w = { 0, 0, 0 };
        if (MODE == 2) {
            const T dtw = (T)st->dt;
#pragma unroll
            for (int jj = 0; jj < S; jj++) { w.x += sa.wcoef[jj] * kj[jj].x; w.y += sa.wcoef[jj] * kj[jj].y; w.z += sa.wcoef[jj] * kj[jj].z; }
            w.x *= dtw; w.y *= dtw; w.z *= dtw;
        }
        T kn2 = 0;
        v3<T> res = stage_result<T, MODE>(lp, mi, H, tau, w, MAXK, &kn2);
        if (!live) { res.x = 0; res.y = 0; res.z = 0; }
        out[q] = res.x; out[N + q] = res.y; out[2 * N + q] = res.z;
        if (MODE >= 1 && (NEXT || ERR)) {
            const T dt = (T)st->dt;
            if (NEXT) {
                v3<T> acc = { sa.coef[S] * res.x, sa.coef[S] * res.y, sa.coef[S] * res.z };
#pragma unroll
                for (int jj = 0; jj < S; jj++) { acc.x += sa.coef[jj] * kj[jj].x; acc.y += sa.coef[jj] * kj[jj].y; acc.z += sa.coef[jj] * kj[jj].z; }
                if (MODE == 2) {
                    const v3<T> wn = { dt * acc.x, dt * acc.y, dt * acc.z };
                    const v3<T> yn = cayley_apply<T>(wn, m0);
                    sa.ynext[q] = yn.x; sa.ynext[N + q] = yn.y; sa.ynext[2 * N + q] = yn.z;
                } else {
                    sa.ynext[q] = m0.x + dt * acc.x; sa.ynext[N + q] = m0.y + dt * acc.y; sa.ynext[2 * N + q] = m0.z + dt * acc.z;
                }
            }
            if (ERR) {
                v3<T> ea = { sa.ecoef[S] * res.x, sa.ecoef[S] * res.y, sa.ecoef[S] * res.z };
#pragma unroll
                for (int jj = 0; jj < S; jj++) { ea.x += sa.ecoef[jj] * kj[jj].x; ea.y += sa.ecoef[jj] * kj[jj].y; ea.z += sa.ecoef[jj] * kj[jj].z; }
                if (live) errn = sqrt((dt * ea.x) * (dt * ea.x) + (dt * ea.y) * (dt * ea.y) + (dt * ea.z) * (dt * ea.z));
            }
        }
        if (MODE == 1 && MAXK && live) kn = sqrt(res.x * res.x + res.y * res.y + res.z * res.z);
        if (MODE == 2 && MAXK && live) kn = kn2;
    }
    if (MODE == 1 && ERR) block_max_bits(norm_bits(errn), &st->err_bits);
    if (MODE >= 1 && MAXK) block_max_bits(norm_bits(kn), &st->maxk_bits);
}

// Neighbour-presence mask, one byte per cell: bit 0..5 = the -x +x -y +y -z +z neighbour is inside the mesh
// and has Ms != 0 (R4).  Rebuilt whenever Ms is set; read by the vectorised stage kernel.
template <typename T>
__global__ void __launch_bounds__(256) nbmask_kernel(Geom g, const T* __restrict__ Ms, unsigned char* __restrict__ nbm)
{
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= g.N) return;
    const int i = (int)(q & (g.nx - 1)), j = (int)((q >> g.lognx) & (g.ny - 1)), k = (int)(q >> (g.lognx + g.logny));
    const long sy = g.nx, sz = (long)g.nx * g.ny;
    unsigned b = 0;
    if (i > 0 && Ms[q - 1] != (T)0) b |= 1u;
    if (i < g.nx - 1 && Ms[q + 1] != (T)0) b |= 2u;
    if (j > 0 && Ms[q - sy] != (T)0) b |= 4u;
    if (j < g.ny - 1 && Ms[q + sy] != (T)0) b |= 8u;
    if (k > 0 && Ms[q - sz] != (T)0) b |= 16u;
    if (k < g.nz - 1 && Ms[q + sz] != (T)0) b |= 32u;
    nbm[q] = (unsigned char)b;
}

// Vectorised form of llg_stage_kernel: one thread owns CPT consecutive cells along x (16 bytes per
// load: 4 fp32 / 2 fp64 cells), so every centre value, every earlier k_j and both outputs move as
// 16-byte accesses; y / z neighbours are 16-byte loads of the neighbouring rows, x neighbours come
// from the thread's own vector plus one scalar on each side.  Same per-cell arithmetic (and
// operation order) as local_field() / ll_torque() in mm_llg.cuh.  Requires nx % CPT == 0.
template <typename T, int CPT> struct alignas(CPT * sizeof(T)) cellvec { T e[CPT]; };
template <typename T, int CPT> __device__ __forceinline__ cellvec<T, CPT> ldc(const T* p) { return *reinterpret_cast<const cellvec<T, CPT>*>(p); }
template <typename T, int CPT> __device__ __forceinline__ void stc(T* p, const cellvec<T, CPT>& v) { *reinterpret_cast<cellvec<T, CPT>*>(p) = v; }

#ifndef MM_STAGEV_THREADS
#define MM_STAGEV_THREADS 128
#endif
#ifndef MM_STAGEV_CPT
#define MM_STAGEV_CPT 2      // fp32 cells per thread (8-byte loads): measured best on B200; fp64 takes 1 (see launch_stage)
#endif
// GEN: cell-based A and / or D: the A_i, D_i of the six neighbours are loaded like the neighbour
// values of m and turned into the harmonic-mean bond values.
template <typename T, int CPT, int MODE, int S, bool NEXT, bool ERR, bool MAXK, bool GEN>
__global__ void __launch_bounds__(MM_STAGEV_THREADS, sizeof(T) == 8 ? 1 : (GEN ? 3 : 4)) llg_stagev_kernel(Geom g, LocalP<T> lp, const T* __restrict__ y, const T* __restrict__ Ms,
                                                         const unsigned char* __restrict__ nbm, const T* __restrict__ Hd, T* __restrict__ out, StageArgs<T> sa, DevState* st)
{
    if (st->done) return;
    typedef cellvec<T, CPT> CV;
    constexpr unsigned ALLNB = CPT == 1 ? 0x3fu : (CPT == 2 ? 0x3f3fu : 0x3f3f3f3fu);
    const long N = g.N;
    const long q = ((long)blockIdx.x * blockDim.x + threadIdx.x) * CPT;
    unsigned long long eb = 0ull, kb = 0ull;      // bit patterns: max keeps a NaN
    if (q < N) {
        const int i0 = (int)(q & (g.nx - 1)), j = (int)((q >> g.lognx) & (g.ny - 1)), k = (int)(q >> (g.lognx + g.logny));
        const CV Msv = ldc<T, CPT>(Ms + q);
        CV m[3], H[3];
#pragma unroll
        for (int c = 0; c < 3; c++) m[c] = ldc<T, CPT>(y + c * N + q);
        if (Hd != nullptr) {
#pragma unroll
            for (int c = 0; c < 3; c++) H[c] = ldc<T, CPT>(Hd + c * N + q);
        } else {
#pragma unroll
            for (int c = 0; c < 3; c++)
#pragma unroll
                for (int e = 0; e < CPT; e++) H[c].e[e] = 0;
        }
        CV kj[S > 0 ? S : 1][3];
#pragma unroll
        for (int jj = 0; jj < S; jj++)
#pragma unroll
            for (int c = 0; c < 3; c++) kj[jj][c] = ldc<T, CPT>(sa.kprev[jj] + c * N + q);
        CV m0[3];
        if (NEXT) {
#pragma unroll
            for (int c = 0; c < 3; c++) m0[c] = ldc<T, CPT>(sa.m0 + c * N + q);
        }
        CV hx[3];      // external field of the thread's cells: per cell (Eq. 35 with H_i) or uniform
        if (lp.Hcell != nullptr && (lp.terms & 8)) {
#pragma unroll
            for (int c = 0; c < 3; c++) hx[c] = ldc<T, CPT>(lp.Hcell + c * N + q);
        } else {
#pragma unroll
            for (int c = 0; c < 3; c++)
#pragma unroll
                for (int e = 0; e < CPT; e++) hx[c].e[e] = lp.hext[c];
        }
        if (GEN && lp.Hth != nullptr) {      // thermal field of the step in progress (Eq. 42)
#pragma unroll
            for (int c = 0; c < 3; c++) {
                const CV t = ldc<T, CPT>(lp.Hth + c * N + q);
#pragma unroll
                for (int e = 0; e < CPT; e++) H[c].e[e] += t.e[e];
            }
        }
        v3<T> tau[CPT];
#pragma unroll
        for (int e = 0; e < CPT; e++) tau[e] = { 0, 0, 0 };
        if ((lp.terms & 3) != 0 || (GEN && MODE >= 1 && lp.stt_on)) {
            // neighbour rows: index clamped to the own row when outside the mesh, then masked
            const long sy = g.nx, szz = (long)g.nx * g.ny;
            const bool oym = j > 0, oyp = j < g.ny - 1, ozm = k > 0, ozp = k < g.nz - 1, oxm = i0 > 0, oxp = i0 + CPT < g.nx;
            const long qym = oym ? q - sy : q, qyp = oyp ? q + sy : q, qzm = ozm ? q - szz : q, qzp = ozp ? q + szz : q;
            const long qxm = oxm ? q - 1 : q, qxp = oxp ? q + CPT : q;
            CV nym[3], nyp[3], nzm[3], nzp[3];
            T xl[3], xr[3];
#pragma unroll
            for (int c = 0; c < 3; c++) {
                nym[c] = ldc<T, CPT>(y + c * N + qym); nyp[c] = ldc<T, CPT>(y + c * N + qyp);
                nzm[c] = ldc<T, CPT>(y + c * N + qzm); nzp[c] = ldc<T, CPT>(y + c * N + qzp);
                xl[c] = y[c * N + qxm]; xr[c] = y[c * N + qxp];
            }
            // cell-based constants of the thread's cells and of their neighbours (index 0 = A, 1 = D)
            CV pc[2], pym[2], pyp[2], pzm[2], pzp[2];
            T pxl[2], pxr[2];
            if (GEN) {
                const T* par[2] = { lp.Acell, lp.Dcell };
#pragma unroll
                for (int t = 0; t < 2; t++) {
                    if (par[t] != nullptr) {
                        pc[t] = ldc<T, CPT>(par[t] + q);
                        pym[t] = ldc<T, CPT>(par[t] + qym); pyp[t] = ldc<T, CPT>(par[t] + qyp);
                        pzm[t] = ldc<T, CPT>(par[t] + qzm); pzp[t] = ldc<T, CPT>(par[t] + qzp);
                        pxl[t] = par[t][qxm]; pxr[t] = par[t][qxp];
                    }
                }
            }
            // neighbour-presence bits of the thread's cells (nbmask_kernel, written when Ms is set):
            // bit 0..5 = -x +x -y +y -z +z present (inside the mesh and Ms != 0)
            unsigned mk = 0;
#pragma unroll
            for (int e = 0; e < CPT; e++) mk |= (unsigned)nbm[q + e] << (8 * e);
            const bool all_present = (mk & ALLNB) == ALLNB;
#pragma unroll
            for (int e = 0; e < CPT; e++) {
                const T Msi = Msv.e[e];
                const T inv = (T)1 / (Msi != (T)0 ? Msi : (T)1);
                const v3<T> mi = { m[0].e[e], m[1].e[e], m[2].e[e] };
                v3<T> nb[6];
                if (e > 0) nb[0] = { m[0].e[e > 0 ? e - 1 : 0], m[1].e[e > 0 ? e - 1 : 0], m[2].e[e > 0 ? e - 1 : 0] };
                else nb[0] = { xl[0], xl[1], xl[2] };
                if (e < CPT - 1) nb[1] = { m[0].e[e < CPT - 1 ? e + 1 : 0], m[1].e[e < CPT - 1 ? e + 1 : 0], m[2].e[e < CPT - 1 ? e + 1 : 0] };
                else nb[1] = { xr[0], xr[1], xr[2] };
                nb[2] = { nym[0].e[e], nym[1].e[e], nym[2].e[e] };
                nb[3] = { nyp[0].e[e], nyp[1].e[e], nyp[2].e[e] };
                nb[4] = { nzm[0].e[e], nzm[1].e[e], nzm[2].e[e] };
                nb[5] = { nzp[0].e[e], nzp[1].e[e], nzp[2].e[e] };
                v3<T> h = { H[0].e[e], H[1].e[e], H[2].e[e] };
                const v3<T> he = { hx[0].e[e], hx[1].e[e], hx[2].e[e] };
                T w[2][6];
                if (GEN) {
                    const T* par[2] = { lp.Acell, lp.Dcell };
#pragma unroll
                    for (int t = 0; t < 2; t++) {
                        if (par[t] != nullptr) {
                            const T ci = pc[t].e[e];
                            w[t][0] = harm<T>(ci, e > 0 ? pc[t].e[e > 0 ? e - 1 : 0] : pxl[t]);
                            w[t][1] = harm<T>(ci, e < CPT - 1 ? pc[t].e[e < CPT - 1 ? e + 1 : 0] : pxr[t]);
                            w[t][2] = harm<T>(ci, pym[t].e[e]); w[t][3] = harm<T>(ci, pyp[t].e[e]);
                            w[t][4] = harm<T>(ci, pzm[t].e[e]); w[t][5] = harm<T>(ci, pzp[t].e[e]);
                        } else {
#pragma unroll
                            for (int b = 0; b < 6; b++) w[t][b] = (T)1;
                        }
                    }
                }
                if (all_present) {      // interior of the magnetic region: no masking arithmetic at all
                    const bool ok[6] = { true, true, true, true, true, true };
                    h = local_field_nb<T, GEN>(lp, inv, mi, nb, ok, h, he, w[0], w[1]);
                    if (GEN && MODE >= 1 && lp.stt_on) tau[e] = stt_tau<T>(lp, mi, nb, ok);
                } else {
                    bool ok[6];
#pragma unroll
                    for (int b = 0; b < 6; b++) ok[b] = (mk >> (8 * e + b)) & 1u;
                    h = local_field_nb<T, GEN>(lp, inv, mi, nb, ok, h, he, w[0], w[1]);
                    if (GEN && MODE >= 1 && lp.stt_on) tau[e] = stt_tau<T>(lp, mi, nb, ok);
                }
                H[0].e[e] = h.x; H[1].e[e] = h.y; H[2].e[e] = h.z;
            }
        } else {
#pragma unroll
            for (int e = 0; e < CPT; e++) {
                const T Msi = Msv.e[e];
                const T inv = (T)1 / (Msi != (T)0 ? Msi : (T)1);
                const v3<T> mi = { m[0].e[e], m[1].e[e], m[2].e[e] };
                v3<T> h = { H[0].e[e], H[1].e[e], H[2].e[e] };
                const v3<T> he = { hx[0].e[e], hx[1].e[e], hx[2].e[e] };
                h = local_field_rest<T>(lp, inv, mi, h, he);
                H[0].e[e] = h.x; H[1].e[e] = h.y; H[2].e[e] = h.z;
            }
        }
        CV res[3];
#pragma unroll
        for (int e = 0; e < CPT; e++) {
            const bool live = Msv.e[e] != (T)0;
            const v3<T> mi = { m[0].e[e], m[1].e[e], m[2].e[e] };
            const v3<T> h = { H[0].e[e], H[1].e[e], H[2].e[e] };
            v3<T> r;
            T kn2 = 0;
            if (GEN) {
                v3<T> w = { 0, 0, 0 };
                if (MODE == 2) {
                    const T dtw = (T)st->dt;
#pragma unroll
                    for (int jj = 0; jj < S; jj++) { w.x += sa.wcoef[jj] * kj[jj][0].e[e]; w.y += sa.wcoef[jj] * kj[jj][1].e[e]; w.z += sa.wcoef[jj] * kj[jj][2].e[e]; }
                    w.x *= dtw; w.y *= dtw; w.z *= dtw;
                }
                v3<T> te = tau[e];
                if (MODE >= 1) { const T fp = stt_pulse<T>(lp, st, sa.cstage); te.x *= fp; te.y *= fp; te.z *= fp; }
                r = stage_result<T, MODE>(lp, mi, h, te, w, MAXK, &kn2);
            } else {
                r = MODE == 0 ? h : ll_torque<T>(lp, mi, h);
            }
            if (!live) { r.x = 0; r.y = 0; r.z = 0; }
            res[0].e[e] = r.x; res[1].e[e] = r.y; res[2].e[e] = r.z;
            if (MODE == 1 && MAXK && live) { const unsigned long long b = norm_bits(sqrt(r.x * r.x + r.y * r.y + r.z * r.z)); kb = b > kb ? b : kb; }
            if (MODE == 2 && MAXK && live) { const unsigned long long b = norm_bits(kn2); kb = b > kb ? b : kb; }
        }
#pragma unroll
        for (int c = 0; c < 3; c++) stc<T, CPT>(out + c * N + q, res[c]);
        if (MODE >= 1 && (NEXT || ERR)) {
            const T dt = (T)st->dt;
            if (NEXT) {
                CV yn[3];
#pragma unroll
                for (int c = 0; c < 3; c++) {
#pragma unroll
                    for (int e = 0; e < CPT; e++) {
                        T acc = sa.coef[S] * res[c].e[e];
#pragma unroll
                        for (int jj = 0; jj < S; jj++) acc += sa.coef[jj] * kj[jj][c].e[e];
                        yn[c].e[e] = MODE == 2 ? dt * acc : m0[c].e[e] + dt * acc;
                    }
                }
                if (MODE == 2) {      // next stage input Q(omega) m0 (Eq. 43, 47)
#pragma unroll
                    for (int e = 0; e < CPT; e++) {
                        const v3<T> wn = { yn[0].e[e], yn[1].e[e], yn[2].e[e] }, mm0 = { m0[0].e[e], m0[1].e[e], m0[2].e[e] };
                        const v3<T> o = cayley_apply<T>(wn, mm0);
                        yn[0].e[e] = o.x; yn[1].e[e] = o.y; yn[2].e[e] = o.z;
                    }
                }
#pragma unroll
                for (int c = 0; c < 3; c++) stc<T, CPT>(sa.ynext + c * N + q, yn[c]);
            }
            if (ERR) {
#pragma unroll
                for (int e = 0; e < CPT; e++) {
                    T ea[3];
#pragma unroll
                    for (int c = 0; c < 3; c++) {
                        ea[c] = sa.ecoef[S] * res[c].e[e];
#pragma unroll
                        for (int jj = 0; jj < S; jj++) ea[c] += sa.ecoef[jj] * kj[jj][c].e[e];
                    }
                    if (Msv.e[e] != (T)0) {
                        const unsigned long long b = norm_bits(sqrt((dt * ea[0]) * (dt * ea[0]) + (dt * ea[1]) * (dt * ea[1]) + (dt * ea[2]) * (dt * ea[2])));
                        eb = b > eb ? b : eb;
                    }
                }
            }
        }
    }
    if (MODE == 1 && ERR) warp_max_bits(eb, &st->err_bits);
    if (MODE >= 1 && MAXK) warp_max_bits(kb, &st->maxk_bits);
}

// Step controller: one thread.  DESIGN.md R8.
__global__ void ctrl_kernel(DevState* st, int is_f64, int adaptive_mode, int thermal, int nstage)
{
    if (st->done) return;
    if (thermal) st->th_step++;
    st->nrhs += nstage;
    double err, maxk;
    if (is_f64) { err = __longlong_as_double((long long)st->err_bits); maxk = __longlong_as_double((long long)st->maxk_bits); }
    else { err = (double)__uint_as_float((unsigned)st->err_bits); maxk = (double)__uint_as_float((unsigned)st->maxk_bits); }
    st->err_bits = 0ull; st->maxk_bits = 0ull;
    st->err = err; st->maxk = maxk;
    const double tol = st->tol, dt = st->dt;
    const bool bad = !(err == err) || !(maxk == maxk);
    const int ok = !bad && (tol <= 0.0 || err <= tol);
    st->accepted = ok;
    st->nsteps++;
    if (bad) st->nan = 1;
    if (ok) { st->t += dt; st->nacc++; } else st->nrej++;
    double dn = dt;
    if (tol > 0.0) {
        double fac = bad ? 0.2 : (err == 0.0 ? 5.0 : 0.9 * pow(tol / err, 0.2));
        fac = fac < 0.2 ? 0.2 : (fac > 5.0 ? 5.0 : fac);
        dn = dt * fac;
    }
    if (adaptive_mode == 0) { st->dt = dn; return; }          // single step: dt_next reported through st->dt
    if (adaptive_mode == 1) {                                   // relax
        if (maxk < st->stop_dmdt || bad) st->done = 1;
        st->dt = dn;
    } else {                                                    // run until t_end
        const double left = st->t_end - st->t;
        if (left <= 1e-12 * fabs(st->t_end) || bad) { st->done = 1; st->dt = dn; }
        else st->dt = dn < left ? dn : left;
    }
}

// On acceptance: m <- y / |y| on cells with Ms > 0 (projection)
template <typename T>
__global__ void __launch_bounds__(256) accept_kernel(long N, const DevState* st, const T* __restrict__ ysol, const T* __restrict__ Ms, T* __restrict__ m, int project)
{
    if (!st->accepted) return;
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= N || Ms[q] == (T)0) return;
    const T x = ysol[q], y = ysol[N + q], z = ysol[2 * N + q];
    const T n = project ? sqrt(x * x + y * y + z * z) : (T)1;      // Cayley steps are rotations: no projection
    m[q] = x / n; m[N + q] = y / n; m[2 * N + q] = z / n;
}

__global__ void set_state_kernel(DevState* st, double dt, double tol, double t_end, double stop, int mode, int reset_done)
{
    st->dt = dt; st->tol = tol; st->t_end = t_end; st->stop_dmdt = stop; st->mode = mode;
    st->err_bits = 0ull; st->maxk_bits = 0ull;
    if (reset_done) { st->done = 0; st->nan = 0; st->nsteps = 0; }      // nacc / nrej / nrhs run on: lifetime totals
}

// per-block partial sums: out[block*4 + {0,1,2,3}] = sum w*a.b (w = Ms or 1), components / count
template <typename T>
__global__ void __launch_bounds__(256) dot_kernel(long N, const T* __restrict__ a, const T* __restrict__ b, const T* __restrict__ Ms, int mode, double* out)
{
    // mode 0: sum Ms * a.b  -> out[4*blk]; mode 1: sums of a.x, a.y, a.z over Ms>0 and the count
    __shared__ double red[4][256];
    double v[4] = { 0, 0, 0, 0 };
    for (long q = (long)blockIdx.x * blockDim.x + threadIdx.x; q < N; q += (long)gridDim.x * blockDim.x) {
        const double w = (double)Ms[q];
        if (w == 0.0) continue;
        if (mode == 0) v[0] += w * ((double)a[q] * (double)b[q] + (double)a[N + q] * (double)b[N + q] + (double)a[2 * N + q] * (double)b[2 * N + q]);
        else { v[0] += (double)a[q]; v[1] += (double)a[N + q]; v[2] += (double)a[2 * N + q]; v[3] += 1.0; }
    }
    for (int c = 0; c < 4; c++) red[c][threadIdx.x] = v[c];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) for (int c = 0; c < 4; c++) red[c][threadIdx.x] += red[c][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) for (int c = 0; c < 4; c++) out[4 * blockIdx.x + c] = red[c][0];
}

// ------------------------------------------------------------------------------------------------
// Steepest-descent minimiser with Barzilai-Borwein steps (Eq. 50-52; R16)
// ------------------------------------------------------------------------------------------------
struct MinState {
    double tau, tau0, tau_min, tau_max, stop, maxg;
    unsigned long long maxg_bits;
    long long iter, max_steps;      // updates done so far / allowed
    int done, nan;
};

// g_k = m x (m x H_eff(m_k)) and f_k^2 per cell (text under Eq. 51); partial sums of Eq. 52 per block in fp64,
// combined in a fixed order (deterministic); max |g_k| by the bit-pattern maximum.
template <typename T>
__global__ void __launch_bounds__(256) sd_field_kernel(Geom g, LocalP<T> lp, const T* __restrict__ m, const T* __restrict__ Ms, const T* __restrict__ Hd,
                                                       T* __restrict__ gcur, const T* __restrict__ gprev, const T* __restrict__ sprev, T* __restrict__ f2,
                                                       double* __restrict__ part, MinState* ms)
{
    if (ms->done) return;
    const long N = g.N;
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    double ss = 0, sy = 0, yy = 0;
    T gn = 0;
    if (q < N) {
        const T Msi = Ms[q];
        v3<T> gk = { 0, 0, 0 };
        T ff = 0;
        if (Msi != (T)0) {
            const int i = (int)(q & (g.nx - 1)), j = (int)((q >> g.lognx) & (g.ny - 1)), k = (int)(q >> (g.lognx + g.logny));
            const v3<T> mi = ld3(m, N, q);
            v3<T> H = { 0, 0, 0 };
            if (Hd != nullptr) H = ld3(Hd, N, q);
            H = local_field<T>(g, lp, m, Ms, i, j, k, q, Msi, mi, H);
            const T fx = mi.y * H.z - mi.z * H.y, fy = mi.z * H.x - mi.x * H.z, fz = mi.x * H.y - mi.y * H.x;       // f = m x H
            gk.x = mi.y * fz - mi.z * fy; gk.y = mi.z * fx - mi.x * fz; gk.z = mi.x * fy - mi.y * fx;               // g = m x f
            ff = fx * fx + fy * fy + fz * fz;
            gn = sqrt(gk.x * gk.x + gk.y * gk.y + gk.z * gk.z);
            if (ms->iter > 0) {
                const v3<T> sv = ld3(sprev, N, q), gp = ld3(gprev, N, q);
                const double yx = (double)(gk.x - gp.x), yyv = (double)(gk.y - gp.y), yz = (double)(gk.z - gp.z);
                ss = (double)sv.x * sv.x + (double)sv.y * sv.y + (double)sv.z * sv.z;
                sy = (double)sv.x * yx + (double)sv.y * yyv + (double)sv.z * yz;
                yy = yx * yx + yyv * yyv + yz * yz;
            }
        }
        gcur[q] = gk.x; gcur[N + q] = gk.y; gcur[2 * N + q] = gk.z;
        f2[q] = ff;
    }
    __shared__ double red[3][256];
    red[0][threadIdx.x] = ss; red[1][threadIdx.x] = sy; red[2][threadIdx.x] = yy;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) for (int c = 0; c < 3; c++) red[c][threadIdx.x] += red[c][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) for (int c = 0; c < 3; c++) part[3 * (long)blockIdx.x + c] = red[c][0];
    block_max_bits(norm_bits(gn), &ms->maxg_bits);
}

// One block: sums the per-block partials in a fixed order, takes the stop decision and the next tau (Eq. 52).
__global__ void __launch_bounds__(256) sd_ctrl_kernel(const double* __restrict__ part, long nblk, int is_f64, MinState* ms)
{
    if (ms->done) return;
    __shared__ double red[3][256];
    double v[3] = { 0, 0, 0 };
    for (long b = threadIdx.x; b < nblk; b += 256) for (int c = 0; c < 3; c++) v[c] += part[3 * b + c];
    for (int c = 0; c < 3; c++) red[c][threadIdx.x] = v[c];
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) for (int c = 0; c < 3; c++) red[c][threadIdx.x] += red[c][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x != 0) return;
    const double maxg = is_f64 ? __longlong_as_double((long long)ms->maxg_bits) : (double)__uint_as_float((unsigned)ms->maxg_bits);
    ms->maxg_bits = 0ull;
    ms->maxg = maxg;
    if (!(maxg == maxg)) { ms->nan = 1; ms->done = 1; return; }
    if (maxg < ms->stop || ms->iter >= ms->max_steps) { ms->done = 1; return; }
    if (ms->iter > 0) {
        const double ss = red[0][0], sy = red[1][0], yy = red[2][0];
        double t = (ms->iter & 1) ? ss / sy : sy / yy;
        t = fabs(t);
        if (!(t > 0.0) || isinf(t)) t = ms->tau0;
        ms->tau = t < ms->tau_min ? ms->tau_min : (t > ms->tau_max ? ms->tau_max : t);
    }
}

// Eq. 51, per cell; keeps s_k = m_{k+1} - m_k for the next Eq. 52.
template <typename T>
__global__ void __launch_bounds__(256) sd_update_kernel(long N, T* __restrict__ m, const T* __restrict__ gcur, const T* __restrict__ f2, const T* __restrict__ Ms,
                                                        T* __restrict__ sprev, MinState* ms)
{
    if (ms->done) return;
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    const T tau = (T)ms->tau;
    if (q < N && Ms[q] != (T)0) {
        const T a = (T)0.25 * tau * tau * f2[q];
#pragma unroll
        for (int c = 0; c < 3; c++) {
            const T mo = m[c * N + q];
            const T mn = (((T)1 - a) * mo - tau * gcur[c * N + q]) / ((T)1 + a);
            m[c * N + q] = mn;
            sprev[c * N + q] = mn - mo;
        }
    }
}
// separate launch: every block of sd_update_kernel must have read ms->iter-independent state before it moves on
__global__ void sd_count_kernel(MinState* ms) { if (!ms->done) ms->iter++; }

// ------------------------------------------------------------------------------------------------
// Thermal field, Eq. 41-42: xi = eta sqrt(2 alpha kB T / (mu0 Ms gamma V dt)), one Gaussian vector
// per cell and step attempt.  eta: Philox4x32-10 on counter (cell lo, cell hi, step lo, step hi), key (seed lo, seed hi);
// the four words x -> u = (x + 1/2) 2^-32; Box-Muller (R18).  Generated in fp64 for both precisions (once
// per step, 3N values), rounded once to the handle's precision.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(unsigned c0, unsigned c1, unsigned c2, unsigned c3, unsigned k0, unsigned k1, unsigned out[4])
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const unsigned lo0 = 0xD2511F53u * c0, hi0 = __umulhi(0xD2511F53u, c0);
        const unsigned lo1 = 0xCD9E8D57u * c2, hi1 = __umulhi(0xCD9E8D57u, c2);
        c0 = hi1 ^ c1 ^ k0; c1 = lo1; c2 = hi0 ^ c3 ^ k1; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// amp2 = 2 alpha kB T / (mu0 gamma V); dt and step < 0: taken from the device controller (the step in progress)
template <typename T>
__global__ void __launch_bounds__(256) thermal_kernel(Geom g, int unx, int uny, const T* __restrict__ Ms, double amp2, unsigned long long seed, double dt_arg, long long step_arg,
                                                      const DevState* st, T* __restrict__ xi)
{
    if (step_arg < 0 && st->done) return;
    const long N = g.N;
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= N) return;
    // Philox counter word = the cell's index in the CALLER's mesh (differs from q when the mesh is embedded)
    const unsigned long long cell = (unsigned long long)((q & (g.nx - 1)) + (long)unx * (((q >> g.lognx) & (g.ny - 1)) + (long)uny * (q >> (g.lognx + g.logny))));
    const double Msi = (double)Ms[q];
    double e0 = 0, e1 = 0, e2 = 0;
    if (Msi != 0.0 && amp2 > 0.0) {
        const double dt = step_arg < 0 ? st->dt : dt_arg;
        const unsigned long long step = step_arg < 0 ? st->th_step : (unsigned long long)step_arg;
        unsigned x[4];
        philox4x32_10((unsigned)cell, (unsigned)(cell >> 32), (unsigned)step, (unsigned)(step >> 32), (unsigned)seed, (unsigned)(seed >> 32), x);
        const double two_pi = 6.283185307179586476925286766559, sc = 1.0 / 4294967296.0;
        const double u0 = ((double)x[0] + 0.5) * sc, u1 = ((double)x[1] + 0.5) * sc, u2 = ((double)x[2] + 0.5) * sc, u3 = ((double)x[3] + 0.5) * sc;
        const double r0 = sqrt(-2.0 * log(u0)), r1 = sqrt(-2.0 * log(u2));
        double sn, cs;
        sincos(two_pi * u1, &sn, &cs);
        const double amp = sqrt(amp2 / (Msi * dt));
        e0 = r0 * cs * amp; e1 = r0 * sn * amp; e2 = r1 * cos(two_pi * u3) * amp;
    }
    xi[q] = (T)e0; xi[N + q] = (T)e1; xi[2 * N + q] = (T)e2;
}

template <typename T> __global__ void fill_kernel(long n, T* p, T v)
{
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q < n) p[q] = v;
}

// ------------------------------------------------------------------------------------------------
// Setup (S0): demag tensor in real space, its spectrum, packing.  fp64 throughout.  PAPER.md:136.
// ------------------------------------------------------------------------------------------------
struct QuadRule { int n[3]; double s[3][32]; double w[3][32]; };

// Far field: N_ab(r) = -(1/(4 pi V)) int_cell int_cell' d_a d_b (1/|r + u - u'|) du du'  — the definition
// of the cell-averaged tensor — by a 5-point Gauss-Legendre rule in each of the six variables,
// collapsed to a rule in the differences s = u - u' (rule.s / rule.w, weights sum to 1 per axis).
// Near box (|offset| < b in every axis): values from the host quad-precision closed forms.
__global__ void __launch_bounds__(128) tensor_real_kernel(int nx, int ny, int nz, double dx, double dy, double dz, QuadRule rule,
                                                          int bx, int by, int bz, const double* __restrict__ near, double* __restrict__ Nr)
{
    const long N = (long)nx * ny * nz;
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= N) return;
    const int i = (int)(q % nx), j = (int)((q / nx) % ny), k = (int)(q / ((long)nx * ny));
    if (i < bx && j < by && k < bz) {
        const long Bn = (long)bx * by * bz, o = i + (long)bx * (j + (long)by * k);
        for (int c = 0; c < 6; c++) Nr[c * N + q] = near[c * Bn + o];
        return;
    }
    const double X = i * dx, Y = j * dy, Z = k * dz;
    double a[6] = { 0, 0, 0, 0, 0, 0 };
    for (int c3 = 0; c3 < rule.n[2]; c3++) {
        const double rz = Z + rule.s[2][c3], wz = rule.w[2][c3];
        for (int b = 0; b < rule.n[1]; b++) {
            const double ry = Y + rule.s[1][b], wyz = wz * rule.w[1][b];
            for (int aa = 0; aa < rule.n[0]; aa++) {
                const double rx = X + rule.s[0][aa], w = wyz * rule.w[0][aa];
                const double r2 = rx * rx + ry * ry + rz * rz;
                const double ir = rsqrt(r2), ir2 = ir * ir, ir5 = ir2 * ir2 * ir * w;
                a[0] += (3.0 * rx * rx - r2) * ir5; a[1] += (3.0 * ry * ry - r2) * ir5; a[2] += (3.0 * rz * rz - r2) * ir5;
                a[3] += 3.0 * rx * ry * ir5; a[4] += 3.0 * rx * rz * ir5; a[5] += 3.0 * ry * rz * ir5;
            }
        }
    }
    const double pref = -(dx * dy * dz) / (4.0 * 3.14159265358979323846264338327950288);
    for (int c = 0; c < 6; c++) Nr[c * N + q] = pref * a[c];
}

// Kernel array on the padded grid with wrap indexing (R3): padded index p is offset p for
// p < n, p - 2n for p > n, slot p = n is 0.  Off-diagonal components are odd in their two axes.
__global__ void __launch_bounds__(256) wrap_kernel(Geom g, int comp, const double* __restrict__ Nr, cx<double>* __restrict__ A)
{
    const long P = (long)g.px * g.py * g.pz;
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= P) return;
    const int a = (int)(q % g.px), b = (int)((q / g.px) % g.py), c = (int)(q / ((long)g.px * g.py));
    double v = 0.0;
    const bool hole = (g.nx > 1 && a == g.nx) || (g.ny > 1 && b == g.ny) || (g.nz > 1 && c == g.nz);
    if (!hole) {
        const int di = a < g.nx ? a : a - g.px, dj = b < g.ny ? b : b - g.py, dk = c < g.nz ? c : c - g.pz;
        const int sx = di < 0 ? -1 : 1, sy = dj < 0 ? -1 : 1, sz = dk < 0 ? -1 : 1;
        const long o = abs(di) + (long)g.nx * (abs(dj) + (long)g.ny * abs(dk));
        v = Nr[comp * g.N + o];
        if (comp == 3) v *= sx * sy;
        if (comp == 4) v *= sx * sz;
        if (comp == 5) v *= sy * sz;
    }
    A[q] = mk<double>(v, 0.0);
}

// Generic batched line FFT (forward DIF, output in bit-reversed positions) used only at setup.
// Line l = (outer, inner): base = outer*so + inner*si ; points stride sp.  One CTA: LT lines.
__global__ void __launch_bounds__(256) setup_fft_kernel(cx<double>* A, int n, long sp, int ninner, long si, long so, int LT, int point_fastest,
                                                        twiddles<double> tw)
{
    cx<double>* s = reinterpret_cast<cx<double>*>(mm_smem);
    const int pitch = odd_pitch(LT);
    const long line0 = (long)blockIdx.x * LT;
    for (int f = threadIdx.x; f < n * LT; f += blockDim.x) {
        const int p = point_fastest ? f % n : f / LT, l = point_fastest ? f / n : f % LT;
        const long line = line0 + l;
        s[(size_t)p * pitch + l] = A[(line / ninner) * so + (line % ninner) * si + (long)p * sp];
    }
    __syncthreads();
    fft_fwd_blocks<double>(s, pitch, LT, n, n, tw, threadIdx.x, blockDim.x);
    for (int f = threadIdx.x; f < n * LT; f += blockDim.x) {
        const int p = point_fastest ? f % n : f / LT, l = point_fastest ? f / n : f % LT;
        const long line = line0 + l;
        A[(line / ninner) * so + (line % ninner) * si + (long)p * sp] = s[(size_t)p * pitch + l];
    }
}

// Symmetric-packed real spectrum in the positions pass B reads: Kh[comp][kz'][ky'][xpos].
// Also accumulates max |Im| and max |Re| (bit patterns) for the "K^ is real" check.
template <typename T>
__global__ void __launch_bounds__(256) pack_khat_kernel(Geom g, int comp, const cx<double>* __restrict__ A, T* __restrict__ Kh, unsigned long long* maxbits)
{
    const int nkz = g.nz > 1 ? g.nz + 1 : 1;
    const long total = (long)nkz * (g.ny + 1) * g.Lx;
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    double re = 0.0, im = 0.0;
    if (q < total) {
        const int xp = (int)(q % g.Lx), kyp = (int)((q / g.Lx) % (g.ny + 1)), kzp = (int)(q / ((long)g.Lx * (g.ny + 1)));
        if (xp <= g.nx) {
            const int kx = xp < g.nx ? (int)brev((unsigned)xp, g.lognx) : g.nx;
            const long a = brev((unsigned)kx, g.lognx + 1), b = brev((unsigned)kyp, g.logpy), c = g.nz > 1 ? brev((unsigned)kzp, g.logpz) : 0;
            const cx<double> v = A[a + (long)g.px * (b + (long)g.py * c)];
            re = v.x; im = v.y;
        }
        Kh[(long)comp * g.kcomp + q] = (T)re;
    }
    block_max_bits(norm_bits(fabs(re)), maxbits);
    block_max_bits(norm_bits(fabs(im)), maxbits + 1);
}

template <typename T> __global__ void __launch_bounds__(256) kc_fill_kernel(Geom g, const T* __restrict__ Kh, T* __restrict__ Kc, long total)
{
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx < total) kc_fill<T>(g, Kh, Kc, idx);
}

}  // namespace mm

// ================================================================================================
// Host runtime
// ================================================================================================
using namespace mm;

static constexpr size_t STEP_KEY_MAX = 256;      // bytes of a step-graph key (step_key)

struct mm_sim {
    Geom g;
    mm_prec prec;
    int device;
    cudaStream_t stream;
    double dx, dy, dz;
    double A, D, Ku, Kc, u[3], hext[3], alpha, gamma;
    int dmi_kind, integ, demag_on, demag_ready, Ms_set;
    int dmi_kind_uniform = 0;                // the kind given to mm_set_D; dmi_kind is the active one (cell-based D carries its own)
    int A_cell, D_cell, H_cell;      // cell-based A / D / external field set (arrays in the workspace)
    int unx, uny, unz, embed;        // the caller's mesh; embed: it is not 2^k per axis and lives inside the padded mesh g
    long uN;
    // whole-step CUDA graphs (one launch per step instead of ~30): captured on the second step with the same key
    struct StepGraph { unsigned char key[STEP_KEY_MAX]; size_t key_len; cudaGraphExec_t exec; long launches; };
    std::vector<StepGraph> graphs;
    cudaStream_t cap_stream;         // capture happens on a private stream (the caller's may be the legacy default stream)
    int use_graph;
    int b7_narrow;                   // fp32, ny = 512 / 1024: the specialised pass B runs tiles of 2 columns, four / two CTAs per SM
    int use_b4, clQ;                 // pass B runs the cluster form with clusters of clQ CTAs (long lines)
    int use_b3;                      // pass B runs the half-tile form (a full py-row tile does not fit one CTA)
    size_t off_S2;                   // its output spectrum
    size_t off_ei, off_eo;           // embedding: inner-layout copies of the caller's input / output fields
    double stt_u[3], stt_beta, stt_b, stt_w, sl_aJ, sl_bJ, sl_p[3], temperature;      // Zhang-Li, Slonczewski / SOT, thermal field
    unsigned long long th_seed;
    // workspace
    void* ws;
    size_t ws_bytes, ws_need;
    size_t off_Ms, off_nbm, off_S, off_Kh, off_Kc, off_mh, off_Hd, off_k[7], off_y[2], off_tw, off_st, off_part, off_min, off_Ac, off_Dc, off_Hc, off_Hth;
    int twN;
    size_t smemA, smemA2, smemB;
    int thrA, thrB;
    double khat_imag_ratio;
    double t_host;
    long launches;
    std::string err;
    // optional per-pass profiling (mm_set_profiling): event pairs around each kernel class
    int use_v2;
    int use_tma;            // pass B moves its tile rows with TMA tensor-map copies
    int no_b7;              // MM_NO_B7: keep the generic TMA pass B (A/B comparisons)
    CUtensorMap tmS;        // S as (x, j, zpos, comp)
    int no_stagev;          // MM_NO_STAGEV: one-cell-per-thread stage kernel (A/B comparisons)
    std::vector<const void*> smem_attr;      // kernels whose dynamic shared-memory limit has been raised on s->device
    bool launch_skipped = false;             // a launch_* helper returned without launching (s->err says why); read by demag_passes
    int prof_on, prof_open;      // prof_on: bit c = kernel class c is bracketed with events
    std::vector<cudaEvent_t> prof_ev;      // pairs
    std::vector<int> prof_cls;             // class of pair i: 0 pass A, 1 pass B, 2 pass C, 3 stage kernel
    size_t prof_used;
};

static const size_t PROF_MAX_PAIRS = 1 << 14;      // brackets kept between two mm_get_profile calls; later kernels run unbracketed
static void prof_begin(mm_sim* s, int cls)
{
    s->prof_open = (s->prof_on >> cls) & 1;
    if (!s->prof_open) return;
    if (s->prof_used >= PROF_MAX_PAIRS) { s->prof_open = 0; return; }
    if (s->prof_used + 1 > s->prof_cls.size()) {
        cudaEvent_t a = nullptr, b = nullptr;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) {
            if (a) cudaEventDestroy(a);
            cudaGetLastError(); s->prof_open = 0; return;
        }
        s->prof_ev.push_back(a); s->prof_ev.push_back(b); s->prof_cls.push_back(cls);
    }
    s->prof_cls[s->prof_used] = cls;
    if (cudaEventRecord(s->prof_ev[2 * s->prof_used], s->stream) != cudaSuccess) { cudaGetLastError(); s->prof_open = 0; }
}
static void prof_end(mm_sim* s)
{
    if (!s->prof_open) return;
    s->prof_open = 0;
    if (cudaEventRecord(s->prof_ev[2 * s->prof_used + 1], s->stream) != cudaSuccess) { cudaGetLastError(); return; }
    s->prof_used++;
}

#define MM_TRY(sim, call)                                                                          \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            (sim)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                       \
            return MM_ERR_CUDA;                                                                    \
        }                                                                                          \
    } while (0)

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device setting: recorded per handle (a handle lives on one
// device), not per process.  Returns false when the driver refuses: the caller then skips its launch, and because the
// CUDA error is consumed here, s->launch_skipped carries the failure to demag_passes, which returns MM_ERR_CUDA
// (message in s->err) instead of reporting a field that was never computed.
static bool raise_smem_limit(mm_sim* s, const void* func)
{
    for (const void* f : s->smem_attr) if (f == func) return true;
    const cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e != cudaSuccess) { s->err = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e); cudaGetLastError(); s->launch_skipped = true; return false; }
    s->smem_attr.push_back(func);
    return true;
}

static int fail(mm_sim* s, int code, const char* msg) { if (s) s->err = msg; return code; }
static size_t esize(const mm_sim* s) { return s->prec == MM_F64 ? sizeof(double) : sizeof(float); }
static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }
static int next_pow2(int v) { int p = 1; while (p < v) p <<= 1; return p; }
template <typename T> static T* wsp(const mm_sim* s, size_t off) { return reinterpret_cast<T*>(static_cast<char*>(s->ws) + off); }
static const size_t SMEM_CAP = 200 * 1024;

// Tile configuration.
static void configure(mm_sim* s)
{
    Geom& g = s->g;
    const size_t cs = 2 * esize(s);
    const int target = 2 * 148;      // minimum grid size aimed at
    // passes A/C: G rows per CTA
    int G = 1;
    if (g.nz < 8) {
        G = 16;
        while (G > 1 && (G > g.ny || 3 * (g.ny / G) < target)) G /= 2;
    }
    g.G = G;
    g.CH = 64;
    if (g.nz > 1) while (g.CH > 8 && (size_t)g.pz * g.G * g.CH * cs > 32 * 1024) g.CH /= 2;
    // at most 4 lines per CTA (long film lines): padded x tile, see ppos() in mm_kernels.cuh (measured: 4096^2 pass A 673 -> 568 us, 2048^2 168 -> 158; with 8 lines it is slower, 1024^2 41 -> 53 us)
    g.xpad = g.G * g.nz <= 4 ? 1 : 0;
    // <= 100 KB: two CTAs per SM (one 200 KB tile per SM measured 15-30 % slower on films of 2048^2 and 4096^2)
    while (g.G > 1 && (size_t)smemA_elems(g) * cs > 100 * 1024) g.G /= 2;
    // pass B: TC columns per CTA
    int TC = s->prec == MM_F64 ? 4 : 8;
    if (getenv("MM_TC")) TC = atoi(getenv("MM_TC"));       // tuning knob (power of two)
    g.TC = TC;
    while (g.TC > 1 && (size_t)smemB_elems(g) * cs > SMEM_CAP) g.TC /= 2;
    // a line that does not fit one CTA even one column wide (fp64, ny = 4096) -> a cluster of Q CTAs shares the line,
    // each with a tile of py/Q rows of 32 bytes (mm_passB4.cuh).  Measured (profiles/r02_experiments.md): 4096^2 fp64
    // 4.2 ms against 5.2 ms of the half-tile form; where a full tile still fits (TC = 2 or 1) the single-CTA kernels
    // stay faster (2048^2 fp32 184 us against 306 / 418 us with clusters of 2 / 4), so they keep those sizes.
    s->use_b4 = 0; s->clQ = 0;
    {
        const int tcmin = s->prec == MM_F64 ? 2 : 4;
        if (s->use_v2 && !getenv("MM_NO_B4") && !getenv("MM_B3") && ((size_t)g.py * 3 * cs > SMEM_CAP || getenv("MM_B4"))) {
            // the smallest cluster whose tile fits, with the widest rows that fit it (measured at 4096^2 fp64: Q = 2 with
            // 16-byte rows 2.9 ms, Q = 4 with 32-byte rows 4.2 ms — every CTA re-reads the whole input line)
            for (int Q = 2; Q <= 4 && !s->use_b4; Q *= 2) {
                if (getenv("MM_Q") && atoi(getenv("MM_Q")) != Q) continue;
                for (int tc = getenv("MM_TC") ? atoi(getenv("MM_TC")) : tcmin; tc >= 1 && !s->use_b4; tc /= 2)
                    if (g.py / Q >= 16 && (size_t)(g.py / Q) * 3 * tc * cs <= SMEM_CAP) { s->use_b4 = 1; s->clQ = Q; g.TC = tc; }
            }
        }
    }
    // a line that does not fit even one column wide (or MM_B3=1, for measurements): half-tile form, ny rows per tile
    s->use_b3 = 0;
    if (!s->use_b4 && s->use_v2 && g.ny >= 16 && ((size_t)smemB_elems(g) * cs > SMEM_CAP || getenv("MM_B3"))) {
        s->use_b3 = 1;
        g.TC = s->prec == MM_F64 ? 4 : 8;
        if (getenv("MM_TC")) g.TC = atoi(getenv("MM_TC"));
        while (g.TC > 1 && (size_t)g.ny * 3 * g.TC * cs > SMEM_CAP) g.TC /= 2;
    }
    // fp32: two resident CTAs per SM (tile <= 98 KB) beat one CTA with a tile twice as wide — one CTA's
    // shared-memory-bound stages overlap the other's FP32-bound ones (measured, profiles/r01_experiments.md)
    if (s->prec == MM_F32 && !getenv("MM_TC") && g.TC >= 4 && (size_t)smemB_elems(g) * cs > 98 * 1024) g.TC /= 2;
    while (g.TC > 2 && ((g.nx + g.TC) / g.TC) * g.pz < target && !s->use_b3 && !s->use_b4) g.TC /= 2;
    // fp64: the specialised pass B (mm_passB7.cuh) wants rows of 32 bytes = two columns, tiles of py * 96 bytes
    const bool b7_f64 = s->prec == MM_F64 && !getenv("MM_TC") && !s->no_b7 && !s->use_b3 && !s->use_b4 && s->use_v2 && g.logny >= 4 && g.logny <= 10 && g.TC >= 2;
    if (b7_f64) g.TC = 2;
    // ny = 1024: the specialised pass B with one 196 KB tile per SM (rows of 32 bytes in both precisions)
    const bool b7_10 = g.logny == 10 && !getenv("MM_TC") && !s->no_b7 && !s->use_b3 && !s->use_b4 && s->use_v2;
    if (b7_10 && s->prec == MM_F32) g.TC = 4;
    s->b7_narrow = (s->prec == MM_F32 && (g.logny == 9 || g.logny == 10) && g.TC == 4 && !getenv("MM_TC") && !s->no_b7 && !s->use_b3 && !s->use_b4 && s->use_v2 && !(getenv("MM_NO_NARROW") && getenv("MM_NO_NARROW")[0])) ? 1 : 0;
    if (s->b7_narrow) g.TC = 2;
    g.Lx = ((g.nx + 1 + g.TC - 1) / g.TC) * g.TC;
    if (s->b7_narrow) g.Lx = ((g.nx + 1 + 3) / 4) * 4;      // rows of S keep their 32-byte alignment for passes A / C
    g.plane = (long)g.ny * g.Lx;
    g.comp = (long)g.pz * g.plane;
    g.kplane = (long)(g.ny + 1) * g.Lx;
    g.kcomp = (long)(g.nz > 1 ? g.nz + 1 : 1) * g.kplane;
    s->smemA = (size_t)smemA_elems(g) * cs;
    // the v2 bodies of passes A / C do the z transform in registers: no scratch tile
    g.xpad = g.G * g.nz <= 4 ? 1 : 0;      // G may have shrunk above
    s->smemA2 = (size_t)smemA2_elems(g) * cs;
    s->smemB = s->use_b4 ? (size_t)smemB4_elems(g, s->clQ) * cs : (s->use_b3 ? (size_t)smemB3_elems(g) * cs : (size_t)smemB_elems(g) * cs);
    s->thrA = 256;
    s->thrB = (s->prec == MM_F32 && s->smemB > 98 * 1024) ? 512 : 256;
    if (b7_f64) s->thrB = 128;
    if (b7_10) s->thrB = s->prec == MM_F64 ? 256 : 512;
    if (s->b7_narrow) s->thrB = g.logny >= 10 ? 256 : 128;
    if (s->use_b4) s->thrB = 256;
    if (s->use_b3) s->thrB = 256;      // 255 registers per thread: the multiply stage holds 3 x 8 complex values + K^ (512 threads spilled kilobytes)
    if (getenv("MM_THRB")) s->thrB = atoi(getenv("MM_THRB"));
}

static void layout(mm_sim* s)
{
    const Geom& g = s->g;
    const size_t es = esize(s), N = (size_t)g.N;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o = align256(o + bytes); return r; };
    s->off_st = take(sizeof(DevState));
    s->off_Ms = take(N * es);
    s->off_nbm = take(N);
    s->off_S = take((size_t)3 * g.comp * 2 * es);
    s->off_S2 = take(s->use_b3 ? (size_t)3 * g.comp * 2 * es : 0);
    s->off_Kh = take((size_t)6 * g.kcomp * es);
    s->off_Kc = take((s->use_v2 && g.ny >= 16 && !s->use_b3 && !s->use_b4 ? (size_t)kc_elems(g) : 0) * es);      // pass B v2: K^ in consumption order
    s->off_Hd = take(3 * N * es);
    for (int i = 0; i < 7; i++) s->off_k[i] = take(3 * N * es);
    for (int i = 0; i < 2; i++) s->off_y[i] = take(3 * N * es);
    s->off_mh = take(3 * N * es);      // staging slot of the host-buffer entry points
    s->off_tw = take((size_t)(s->twN / 2 + 1) * 2 * es);
    s->off_part = take(3 * (size_t)((N + 255) / 256) * sizeof(double) > 4 * 1024 * sizeof(double) ? 3 * (size_t)((N + 255) / 256) * sizeof(double) : 4 * 1024 * sizeof(double));
    s->off_min = take(sizeof(MinState));
    s->off_Ac = take(N * es);          // cell-based A_i, D_i, H_ext,i (Eq. 35): 5N reals
    s->off_Dc = take(N * es);
    s->off_Hc = take(3 * N * es);
    s->off_Hth = take(3 * N * es);     // thermal field of the step in progress (Eq. 42)
    s->off_ei = take(s->embed ? 3 * N * es : 0);
    s->off_eo = take(s->embed ? 3 * N * es : 0);
    s->ws_need = o;
}

extern "C" const char* mm_version(void) { return "mm-b200 0.4 (sm_100a)"; }

extern "C" int mm_create(mm_sim** out, int nx, int ny, int nz, double dx, double dy, double dz, mm_prec prec, int device, void* cuda_stream)
{
    if (!out) return MM_ERR_ARG;
    *out = nullptr;
    if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || (prec != MM_F32 && prec != MM_F64)) return MM_ERR_ARG;
    // Any mesh size: a size that is not a power of two is embedded in the next power of two with vacuum (Ms = 0) cells
    // — the FFT passes are radix-2 and zero padding beyond 2n - 1 does not change the convolution (R3); the
    // caller keeps its own nx x ny x nz layout, the library packs / unpacks at the ABI.
    const int unx = nx, uny = ny, unz = nz;
    if (nx > (1 << 20) || ny > (1 << 20) || nz > (1 << 20)) return MM_ERR_UNSUPPORTED;
    nx = next_pow2(nx); ny = next_pow2(ny); nz = next_pow2(nz);
    if ((long)nx * ny * nz > (1L << 30)) return MM_ERR_UNSUPPORTED;
    mm_sim* s = new mm_sim();
    s->cap_stream = nullptr; s->use_graph = getenv("MM_NO_GRAPH") ? 0 : 1;
    s->unx = unx; s->uny = uny; s->unz = unz; s->uN = (long)unx * uny * unz;
    s->embed = (unx != nx || uny != ny || unz != nz) ? 1 : 0;
    s->prec = prec; s->device = device; s->stream = static_cast<cudaStream_t>(cuda_stream);
    s->dx = dx; s->dy = dy; s->dz = dz;
    s->A = s->D = s->Ku = s->Kc = 0; s->A_cell = s->D_cell = s->H_cell = 0;
    s->stt_u[0] = s->stt_u[1] = s->stt_u[2] = s->stt_beta = 0; s->stt_b = s->stt_w = 0; s->sl_aJ = s->sl_bJ = 0; s->sl_p[0] = s->sl_p[1] = 0; s->sl_p[2] = 1; s->temperature = 0; s->th_seed = 0; s->u[0] = s->u[1] = 0; s->u[2] = 1; s->hext[0] = s->hext[1] = s->hext[2] = 0;
    s->alpha = 0.5; s->gamma = 2.211e5; s->dmi_kind = 0; s->integ = MM_DOPRI5; s->demag_on = 1; s->demag_ready = 0; s->Ms_set = 0;
    s->ws = nullptr; s->ws_bytes = 0; s->khat_imag_ratio = -1; s->t_host = 0; s->launches = 0; s->prof_on = 0; s->prof_open = 0; s->prof_used = 0; s->use_v2 = getenv("MM_FORCE_V1") ? 0 : 1; s->no_b7 = getenv("MM_NO_B7") ? 1 : 0; s->no_stagev = getenv("MM_NO_STAGEV") ? 1 : 0;
    Geom& g = s->g;
    memset(&g, 0, sizeof(g));
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.px = nx > 1 ? 2 * nx : 1; g.py = ny > 1 ? 2 * ny : 1; g.pz = nz > 1 ? 2 * nz : 1;
    g.lognx = ilog2(nx); g.logny = ilog2(ny); g.logpy = ilog2(g.py); g.logpz = ilog2(g.pz);
    g.N = (long)nx * ny * nz;
    s->twN = g.px > g.py ? g.px : g.py;
    if (g.pz > s->twN) s->twN = g.pz;
    if (s->twN < 4) s->twN = 4;
    configure(s);
    if (getenv("MM_FLAGS")) g.flags = atoi(getenv("MM_FLAGS"));
    layout(s);
    *out = s;
    return MM_OK;
}

extern "C" int mm_destroy(mm_sim* s)
{
    if (s) {
        if (s->ws && !s->graphs.empty()) { cudaSetDevice(s->device); cudaStreamSynchronize(s->stream); cudaGetLastError(); }      // no replay in flight
        for (cudaEvent_t e : s->prof_ev) cudaEventDestroy(e);
        for (auto& g : s->graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
        if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    }
    delete s;
    return MM_OK;
}

extern "C" int mm_set_profiling(mm_sim* s, int on)
{
    if (!s) return MM_ERR_ARG;
    s->prof_on = on == 1 ? 15 : ((on >> 1) & 15);      // 1 = all four classes, otherwise bit c+1 = class c
    s->prof_used = 0;
    return MM_OK;
}

extern "C" int mm_get_profile(mm_sim* s, double ms_out[4], long count_out[4])
{
    if (!s || !ms_out || !count_out) return MM_ERR_ARG;
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    for (int c = 0; c < 4; c++) { ms_out[c] = 0; count_out[c] = 0; }
    for (size_t i = 0; i < s->prof_used; i++) {
        float ms = 0;
        MM_TRY(s, cudaEventElapsedTime(&ms, s->prof_ev[2 * i], s->prof_ev[2 * i + 1]));
        ms_out[s->prof_cls[i]] += ms;
        count_out[s->prof_cls[i]]++;
    }
    s->prof_used = 0;
    return MM_OK;
}
extern "C" size_t mm_workspace_bytes(const mm_sim* s) { return s ? s->ws_need : 0; }
extern "C" const char* mm_last_error(const mm_sim* s) { return s ? s->err.c_str() : "null handle"; }
extern "C" long mm_launch_count(const mm_sim* s) { return s ? s->launches : 0; }

template <typename T> static int upload_twiddles(mm_sim* s)
{
    const int n = s->twN / 2 + 1;
    std::vector<cx<T>> h(n);
    for (int k = 0; k < n; k++) {
        const long double a = -2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)s->twN;
        h[k].x = (T)cosl(a); h[k].y = (T)sinl(a);
    }
    // exact values at the octants
    h[0].x = 1; h[0].y = 0;
    if (s->twN % 4 == 0) { h[s->twN / 4].x = 0; h[s->twN / 4].y = -1; }
    h[s->twN / 2].x = -1; h[s->twN / 2].y = 0;
    MM_TRY(s, cudaMemcpyAsync(wsp<char>(s, s->off_tw), h.data(), n * sizeof(cx<T>), cudaMemcpyHostToDevice, s->stream));
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    return MM_OK;
}

extern "C" int mm_set_workspace(mm_sim* s, void* dev_ptr, size_t bytes)
{
    if (!s || !dev_ptr) return MM_ERR_ARG;
    if (bytes < s->ws_need) return fail(s, MM_ERR_NOMEM, "workspace smaller than mm_workspace_bytes()");
    if ((uintptr_t)dev_ptr & 255) return fail(s, MM_ERR_ARG, "workspace must be 256-byte aligned");
    MM_TRY(s, cudaSetDevice(s->device));
    s->ws = dev_ptr; s->ws_bytes = bytes;
    // zero state, Ms and the spectrum (pad columns of S are never written by pass A)
    MM_TRY(s, cudaMemsetAsync(dev_ptr, 0, s->off_Kh, s->stream));
    s->demag_ready = 0; s->Ms_set = 0; s->A_cell = s->D_cell = s->H_cell = 0;
    return s->prec == MM_F64 ? upload_twiddles<double>(s) : upload_twiddles<float>(s);
}

#define NEED_WS(s) do { if (!(s)) return MM_ERR_ARG; if (!(s)->ws) return fail((s), MM_ERR_STATE, "mm_set_workspace not called"); } while (0)

static int build_nbmask(mm_sim* s)
{
    const long N = s->g.N;
    const unsigned blocks = (unsigned)((N + 255) / 256);
    if (s->prec == MM_F64) nbmask_kernel<double><<<blocks, 256, 0, s->stream>>>(s->g, wsp<double>(s, s->off_Ms), wsp<unsigned char>(s, s->off_nbm));
    else nbmask_kernel<float><<<blocks, 256, 0, s->stream>>>(s->g, wsp<float>(s, s->off_Ms), wsp<unsigned char>(s, s->off_nbm));
    s->launches++;
    MM_TRY(s, cudaGetLastError());
    return MM_OK;
}

static int in_set_Ms_uniform(mm_sim* s, double Ms)
{
    NEED_WS(s);
    if (!(Ms >= 0)) return fail(s, MM_ERR_ARG, "Ms must be >= 0");
    const long N = s->g.N;
    const int blocks = (int)((N + 255) / 256);
    if (s->prec == MM_F64) fill_kernel<double><<<blocks, 256, 0, s->stream>>>(N, wsp<double>(s, s->off_Ms), Ms);
    else fill_kernel<float><<<blocks, 256, 0, s->stream>>>(N, wsp<float>(s, s->off_Ms), (float)Ms);
    s->launches++;
    MM_TRY(s, cudaGetLastError());
    { int rc = build_nbmask(s); if (rc) return rc; }
    s->Ms_set = 1;
    return MM_OK;
}
static int in_set_Ms(mm_sim* s, const void* dev_Ms)
{
    NEED_WS(s);
    if (!dev_Ms) return MM_ERR_ARG;
    MM_TRY(s, cudaMemcpyAsync(wsp<char>(s, s->off_Ms), dev_Ms, s->g.N * esize(s), cudaMemcpyDeviceToDevice, s->stream));
    { int rc = build_nbmask(s); if (rc) return rc; }
    s->Ms_set = 1;
    return MM_OK;
}
extern "C" int mm_set_A(mm_sim* s, double A) { if (!s) return MM_ERR_ARG; s->A = A; s->A_cell = 0; return MM_OK; }
extern "C" int mm_set_D(mm_sim* s, double D, mm_dmi_kind kind)
{
    if (!s || kind < 0 || kind > 3) return MM_ERR_ARG;
    s->D = D; s->dmi_kind = s->dmi_kind_uniform = kind; s->D_cell = 0; return MM_OK;
}
// cell-based constants: copied into the workspace; NULL switches back to the uniform value
static int set_cell_array(mm_sim* s, size_t off, size_t count, const void* dev_src, int* flag)
{
    NEED_WS(s);
    if (!dev_src) { *flag = 0; return MM_OK; }
    MM_TRY(s, cudaMemcpyAsync(wsp<char>(s, off), dev_src, count * esize(s), cudaMemcpyDeviceToDevice, s->stream));
    *flag = 1;
    return MM_OK;
}
static int in_set_A_cell(mm_sim* s, const void* dev_A) { if (!s) return MM_ERR_ARG; return set_cell_array(s, s->off_Ac, (size_t)s->g.N, dev_A, &s->A_cell); }
static int in_set_D_cell(mm_sim* s, const void* dev_D, mm_dmi_kind kind)
{
    if (!s || kind < 0 || kind > 3) return MM_ERR_ARG;
    // `kind` belongs to the cell-based D: it is committed only once the array has been copied.  NULL switches back to
    // the uniform D of mm_set_D together with that call's kind; a failed call changes nothing.
    const int rc = set_cell_array(s, s->off_Dc, (size_t)s->g.N, dev_D, &s->D_cell);
    if (rc == MM_OK) s->dmi_kind = dev_D ? (int)kind : s->dmi_kind_uniform;
    return rc;
}
static int in_set_H_ext_cell(mm_sim* s, const void* dev_H) { if (!s) return MM_ERR_ARG; return set_cell_array(s, s->off_Hc, 3 * (size_t)s->g.N, dev_H, &s->H_cell); }
extern "C" int mm_set_Ku(mm_sim* s, double Ku) { if (!s) return MM_ERR_ARG; s->Ku = Ku; return MM_OK; }
extern "C" int mm_set_Kc(mm_sim* s, double Kc) { if (!s) return MM_ERR_ARG; s->Kc = Kc; return MM_OK; }
extern "C" int mm_set_axis(mm_sim* s, double ux, double uy, double uz)
{
    if (!s) return MM_ERR_ARG;
    const double n = sqrt(ux * ux + uy * uy + uz * uz);
    if (!(n > 0)) return fail(s, MM_ERR_ARG, "zero anisotropy axis");
    s->u[0] = ux / n; s->u[1] = uy / n; s->u[2] = uz / n; return MM_OK;
}
extern "C" int mm_set_H_ext(mm_sim* s, double hx, double hy, double hz) { if (!s) return MM_ERR_ARG; s->hext[0] = hx; s->hext[1] = hy; s->hext[2] = hz; return MM_OK; }
extern "C" int mm_set_alpha(mm_sim* s, double a) { if (!s || !(a >= 0)) return MM_ERR_ARG; s->alpha = a; return MM_OK; }
extern "C" int mm_set_gamma(mm_sim* s, double g) { if (!s) return MM_ERR_ARG; s->gamma = g; return MM_OK; }
extern "C" int mm_set_integrator(mm_sim* s, mm_integrator i) { if (!s || (i != MM_RK4 && i != MM_DOPRI5 && i != MM_CAYLEY_RK4)) return MM_ERR_ARG; s->integ = i; return MM_OK; }
extern "C" int mm_set_zhang_li(mm_sim* s, double ux, double uy, double uz, double beta)
{
    if (!s) return MM_ERR_ARG;
    s->stt_u[0] = ux; s->stt_u[1] = uy; s->stt_u[2] = uz; s->stt_beta = beta;
    return MM_OK;
}
extern "C" int mm_set_zhang_li_pulse(mm_sim* s, double b, double w)
{
    if (!s) return MM_ERR_ARG;
    s->stt_b = b; s->stt_w = w;
    return MM_OK;
}
extern "C" int mm_set_slonczewski(mm_sim* s, double aJ, double bJ, double px, double py, double pz)
{
    if (!s) return MM_ERR_ARG;
    const double n = sqrt(px * px + py * py + pz * pz);
    if ((aJ != 0.0 || bJ != 0.0) && !(n > 0)) return fail(s, MM_ERR_ARG, "zero polarisation vector");
    s->sl_aJ = aJ; s->sl_bJ = bJ;
    if (n > 0) { s->sl_p[0] = px / n; s->sl_p[1] = py / n; s->sl_p[2] = pz / n; }
    return MM_OK;
}
extern "C" int mm_set_temperature(mm_sim* s, double T, unsigned long long seed)
{
    NEED_WS(s);
    if (!(T >= 0)) return MM_ERR_ARG;
    s->temperature = T; s->th_seed = seed;
    const unsigned long long zero = 0;
    MM_TRY(s, cudaMemcpyAsync(reinterpret_cast<char*>(wsp<DevState>(s, s->off_st)) + offsetof(DevState, th_step), &zero, sizeof(zero), cudaMemcpyHostToDevice, s->stream));
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    return MM_OK;
}
extern "C" int mm_set_demag(mm_sim* s, int on) { if (!s) return MM_ERR_ARG; s->demag_on = on ? 1 : 0; return MM_OK; }

// ------------------------------------------------------------------------------------------------
// mm_init_demag
// ------------------------------------------------------------------------------------------------
static void make_rule(double d, int* n_out, double* s_out, double* w_out)
{
    // 5-point Gauss-Legendre on [-d/2, d/2] for u and u'; rule for s = u - u' with merged nodes
    static const double x5[5] = { -0.9061798459386640, -0.5384693101056831, 0.0, 0.5384693101056831, 0.9061798459386640 };
    static const double w5[5] = { 0.2369268850561891, 0.4786286704993665, 0.5688888888888889, 0.4786286704993665, 0.2369268850561891 };
    int n = 0;
    for (int a = 0; a < 5; a++)
        for (int b = 0; b < 5; b++) {
            const double sv = (x5[a] - x5[b]) * d / 2, wv = w5[a] * w5[b] / 4;
            int hit = -1;
            for (int k = 0; k < n; k++) if (fabs(s_out[k] - sv) < 1e-13 * d) hit = k;
            if (hit >= 0) w_out[hit] += wv; else { s_out[n] = sv; w_out[n] = wv; n++; }
        }
    *n_out = n;
}

// device scratch that is released on every exit path
struct DevBuf {
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes); }
    template <typename U> U* as() const { return static_cast<U*>(p); }
};

// Real-space tensor N_ab(r) at offsets i, j, k >= 0 (6 components x N doubles) into Nr.
static int build_real_tensor(mm_sim* s, double* Nr)
{
    const Geom& g = s->g;
    cudaStream_t st = s->stream;
    // near box: 8 largest-cell-edges in every direction (quadrature error there < 1e-16)
    const double dmax = fmax(s->dx, fmax(s->dy, s->dz));
    const int bx = (int)fmin((double)g.nx, ceil(8.0 * dmax / s->dx)), by = (int)fmin((double)g.ny, ceil(8.0 * dmax / s->dy)),
              bz = (int)fmin((double)g.nz, ceil(8.0 * dmax / s->dz));
    const size_t Bn = (size_t)bx * by * bz;
    std::vector<double> near(6 * Bn);
    mm_newell_near_box(bx, by, bz, s->dx, s->dy, s->dz, near.data());
    DevBuf d_near;
    MM_TRY(s, d_near.alloc(6 * Bn * sizeof(double)));
    MM_TRY(s, cudaMemcpyAsync(d_near.p, near.data(), 6 * Bn * sizeof(double), cudaMemcpyHostToDevice, st));
    QuadRule rule;
    make_rule(s->dx, &rule.n[0], rule.s[0], rule.w[0]);
    make_rule(s->dy, &rule.n[1], rule.s[1], rule.w[1]);
    make_rule(s->dz, &rule.n[2], rule.s[2], rule.w[2]);
    tensor_real_kernel<<<(unsigned)((g.N + 127) / 128), 128, 0, st>>>(g.nx, g.ny, g.nz, s->dx, s->dy, s->dz, rule, bx, by, bz, d_near.as<double>(), Nr);
    s->launches++;
    MM_TRY(s, cudaGetLastError());
    MM_TRY(s, cudaStreamSynchronize(st));      // d_near and `near` are released on return
    return MM_OK;
}

template <typename T> static int init_demag_t(mm_sim* s)
{
    const Geom& g = s->g;
    const long N = g.N, P = (long)g.px * g.py * g.pz;
    cudaStream_t st = s->stream;
    // Transient arrays.  The padded complex tensor A (P fp64 complex numbers, 128 N bytes at most) lives in the
    // caller's workspace, in the slots of H_d and the RK stage vectors (11 x 3N reals >= 132 N bytes), which hold
    // nothing before the first evaluation; the real-space tensor (6N doubles) and three small tables are
    // cudaMalloc'ed here and freed on every exit path.
    if ((size_t)P * sizeof(cx<double>) > s->off_tw - s->off_Hd) return fail(s, MM_ERR_NOMEM, "workspace scratch smaller than the padded tensor");
    cx<double>* A = wsp<cx<double>>(s, s->off_Hd);
    DevBuf d_Nr, d_max, d_tw;
    MM_TRY(s, d_Nr.alloc((size_t)6 * N * sizeof(double)));
    MM_TRY(s, d_max.alloc(2 * sizeof(unsigned long long)));
    MM_TRY(s, cudaMemsetAsync(d_max.p, 0, 2 * sizeof(unsigned long long), st));
    double* Nr = d_Nr.as<double>();
    { int rc = build_real_tensor(s, Nr); if (rc) return rc; }
    // fp64 twiddles for the setup transforms
    const int twN = s->twN, ntw = twN / 2 + 1;
    std::vector<cx<double>> htw(ntw);
    for (int k = 0; k < ntw; k++) {
        const long double a = -2.0L * 3.14159265358979323846264338327950288L * (long double)k / (long double)twN;
        htw[k].x = (double)cosl(a); htw[k].y = (double)sinl(a);
    }
    MM_TRY(s, d_tw.alloc(ntw * sizeof(cx<double>)));
    MM_TRY(s, cudaMemcpyAsync(d_tw.p, htw.data(), ntw * sizeof(cx<double>), cudaMemcpyHostToDevice, st));
    twiddles<double> tw; tw.tw = d_tw.as<cx<double>>(); tw.twN = twN;
    MM_TRY(s, cudaFuncSetAttribute(setup_fft_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_CAP));
    T* Kh = wsp<T>(s, s->off_Kh);
    MM_TRY(s, cudaMemsetAsync(Kh, 0, (size_t)6 * g.kcomp * sizeof(T), st));
    auto line_fft = [&](int n, long sp, long nlines, int ninner, long si, long so, int pf) -> int {
        if (n <= 1) return MM_OK;
        int LT = 8;
        while (LT > 1 && ((size_t)n * odd_pitch(LT) * sizeof(cx<double>) > SMEM_CAP || nlines % LT || ninner % LT)) LT /= 2;
        const size_t sm = (size_t)n * odd_pitch(LT) * sizeof(cx<double>);
        if (sm > SMEM_CAP) return fail(s, MM_ERR_UNSUPPORTED, "setup FFT line does not fit in shared memory");
        setup_fft_kernel<<<(unsigned)(nlines / LT), 256, sm, st>>>(A, n, sp, ninner, si, so, LT, pf, tw);
        s->launches++;
        MM_TRY(s, cudaGetLastError());
        return MM_OK;
    };
    const int ncomp = g.nz > 1 ? 6 : 4;
    for (int c = 0; c < ncomp; c++) {
        wrap_kernel<<<(unsigned)((P + 255) / 256), 256, 0, st>>>(g, c, Nr, A);
        s->launches++;
        int rc;
        if ((rc = line_fft(g.px, 1, (long)g.py * g.pz, g.py * g.pz, g.px, 0, 1))) return rc;
        if ((rc = line_fft(g.py, g.px, (long)g.px * g.pz, g.px, 1, (long)g.px * g.py, 0))) return rc;
        if ((rc = line_fft(g.pz, (long)g.px * g.py, (long)g.px * g.py, g.px * g.py, 1, 0, 0))) return rc;
        const long total = g.kcomp;
        pack_khat_kernel<T><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(g, c, A, Kh, d_max.as<unsigned long long>());
        s->launches++;
        MM_TRY(s, cudaGetLastError());
    }
    if (s->use_v2 && g.ny >= 16 && !s->use_b3 && !s->use_b4) {
        const long total = kc_elems(g);
        kc_fill_kernel<T><<<(unsigned)((total + 255) / 256), 256, 0, st>>>(g, Kh, wsp<T>(s, s->off_Kc), total);
        s->launches++;
        MM_TRY(s, cudaGetLastError());
    }
    unsigned long long hmax[2];
    MM_TRY(s, cudaMemcpyAsync(hmax, d_max.p, sizeof(hmax), cudaMemcpyDeviceToHost, st));
    MM_TRY(s, cudaStreamSynchronize(st));
    double re, im;
    memcpy(&re, &hmax[0], 8); memcpy(&im, &hmax[1], 8);
    s->khat_imag_ratio = re > 0 ? im / re : -1;
    // a numerical self-check, not a CUDA failure: every component is even, or odd in exactly two axes, so K^ is real
    if (!(s->khat_imag_ratio < 1e-10)) return fail(s, MM_ERR_INTERNAL, "demag tensor spectrum is not real: setup failed its symmetry check");
    return MM_OK;
}

static int make_tmap(mm_sim* s);

extern "C" int mm_init_demag(mm_sim* s)
{
    NEED_WS(s);
    const Geom& g = s->g;
    if (g.nx < 4 || g.ny < 2) return fail(s, MM_ERR_UNSUPPORTED, "demag needs nx >= 4 and ny >= 2");
    if (s->smemA > SMEM_CAP || s->smemB > SMEM_CAP) return fail(s, MM_ERR_UNSUPPORTED, "mesh too large for the shared-memory tiles (DESIGN.md Limits)");
    if (g.nz > 1 && (size_t)g.pz * g.G * g.CH * 2 * esize(s) > 64 * 1024) return fail(s, MM_ERR_UNSUPPORTED, "nz too large");
    MM_TRY(s, cudaSetDevice(s->device));
    int rc = s->prec == MM_F64 ? init_demag_t<double>(s) : init_demag_t<float>(s);
    if (rc) return rc;
    if (s->prec == MM_F64) {
        MM_TRY(s, cudaFuncSetAttribute(fwd_xz_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_CAP));
        MM_TRY(s, cudaFuncSetAttribute(y_conv_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_CAP));
        MM_TRY(s, cudaFuncSetAttribute(inv_zx_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_CAP));
    } else {
        MM_TRY(s, cudaFuncSetAttribute(fwd_xz_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_CAP));
        MM_TRY(s, cudaFuncSetAttribute(y_conv_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_CAP));
        MM_TRY(s, cudaFuncSetAttribute(inv_zx_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_CAP));
    }
    if ((rc = make_tmap(s))) return rc;
    s->demag_ready = 1;
    return MM_OK;
}

static int in_get_demag_kernel(mm_sim* s, int comp, void* dev_out)
{
    NEED_WS(s);
    if (!s->demag_ready) return fail(s, MM_ERR_STATE, "mm_init_demag not called");
    if (comp < 0 || comp > 5 || !dev_out) return MM_ERR_ARG;
    // a test hook, off every hot path: the tensor is not kept resident (6N doubles), it is rebuilt on request
    MM_TRY(s, cudaSetDevice(s->device));
    DevBuf d_Nr;
    MM_TRY(s, d_Nr.alloc((size_t)6 * s->g.N * sizeof(double)));
    int rc = build_real_tensor(s, d_Nr.as<double>());
    if (rc) return rc;
    MM_TRY(s, cudaMemcpyAsync(dev_out, d_Nr.as<double>() + (size_t)comp * s->g.N, s->g.N * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    return MM_OK;
}

// ------------------------------------------------------------------------------------------------
// Field / RHS evaluation
// ------------------------------------------------------------------------------------------------
static const double KB = 1.380649e-23;      // J/K (exact, SI 2019)
static bool thermal_on(const mm_sim* s) { return s->temperature > 0.0 && s->alpha > 0.0; }

// in_step: the evaluation belongs to a time step (the thermal field of that step is part of the field)
template <typename T> static LocalP<T> make_local(const mm_sim* s, int terms, bool in_step = false)
{
    LocalP<T> lp;
    const double d[3] = { s->dx, s->dy, s->dz };
    for (int a = 0; a < 3; a++) {
        lp.cex[a] = (T)(2.0 * (s->A_cell ? 1.0 : s->A) / (MU0 * d[a] * d[a]));
        lp.cdm[a] = (T)((s->D_cell ? 1.0 : s->D) / (MU0 * d[a]));
        lp.u[a] = (T)s->u[a];
        lp.hext[a] = (T)s->hext[a];
    }
    lp.Acell = s->A_cell ? wsp<T>(s, s->off_Ac) : (const T*)nullptr;
    lp.Dcell = s->D_cell ? wsp<T>(s, s->off_Dc) : (const T*)nullptr;
    lp.Hcell = s->H_cell ? wsp<T>(s, s->off_Hc) : (const T*)nullptr;
    lp.cku = (T)(2.0 * s->Ku / MU0);
    lp.ckc = (T)(4.0 * s->Kc / MU0);
    lp.Hth = in_step && thermal_on(s) ? wsp<T>(s, s->off_Hth) : (const T*)nullptr;
    for (int a = 0; a < 3; a++) { lp.stt[a] = (T)(s->stt_u[a] / (2.0 * d[a])); lp.p[a] = (T)s->sl_p[a]; }
    lp.beta = (T)s->stt_beta;
    lp.sl_a = (T)(s->sl_aJ / s->gamma); lp.sl_b = (T)(s->sl_bJ / s->gamma);
    lp.gam = (T)s->gamma; lp.al = (T)s->alpha;
    lp.stt_b = s->stt_b; lp.stt_w = s->stt_w;
    lp.stt_on = (s->stt_u[0] != 0.0 || s->stt_u[1] != 0.0 || s->stt_u[2] != 0.0) ? 1 : 0;
    lp.sl_on = (s->sl_aJ != 0.0 || s->sl_bJ != 0.0) ? 1 : 0;
    lp.gp = (T)(s->gamma / (1.0 + s->alpha * s->alpha));
    lp.agp = (T)(s->alpha * s->gamma / (1.0 + s->alpha * s->alpha));
    lp.dmi = s->dmi_kind;
    lp.terms = terms;
    if (s->A == 0.0 && !s->A_cell) lp.terms &= ~1;
    if ((s->D == 0.0 && !s->D_cell) || s->dmi_kind == 0) lp.terms &= ~2;
    if (s->Ku == 0.0) lp.terms &= ~4;
    if (s->Kc == 0.0) lp.terms &= ~32;
    return lp;
}

// demag passes A, B, C: y -> Hd.  v2 kernels where the mesh allows, v1 otherwise (tiny meshes).
template <typename T, int NZ> static void launch_A2(mm_sim* s, unsigned grid, const T* y, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    // the padded x tile exists only for nz <= 4 (at most 4 lines per CTA)
    if (NZ <= 4 && s->g.xpad) {
        if (!raise_smem_limit(s, (const void*)fwd_xz2_kernel<T, NZ, (NZ <= 4)>)) return;
        fwd_xz2_kernel<T, NZ, (NZ <= 4)><<<grid, s->thrA, s->smemA2, s->stream>>>(s->g, y, wsp<T>(s, s->off_Ms), S, tw, st);
        return;
    }
    if (!raise_smem_limit(s, (const void*)fwd_xz2_kernel<T, NZ, false>)) return;
    fwd_xz2_kernel<T, NZ, false><<<grid, s->thrA, s->smemA2, s->stream>>>(s->g, y, wsp<T>(s, s->off_Ms), S, tw, st);
}
template <typename T, int V, int Q> static void launch_B4(mm_sim* s, unsigned ntile, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    if (!raise_smem_limit(s, (const void*)y_conv4_kernel<T, V, Q>)) return;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = dim3(ntile * Q); cfg.blockDim = dim3(s->thrB); cfg.dynamicSmemBytes = s->smemB; cfg.stream = s->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = Q; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, y_conv4_kernel<T, V, Q>, s->g, S, (const T*)wsp<T>(s, s->off_Kh), tw, st);
    if (e != cudaSuccess) { s->err = std::string("cudaLaunchKernelEx(y_conv4): ") + cudaGetErrorString(e); cudaGetLastError(); s->launch_skipped = true; }
}
template <typename T, int V> static void launch_B3(mm_sim* s, unsigned grid, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    if (!raise_smem_limit(s, (const void*)y_conv3_kernel<T, V>)) return;
    y_conv3_kernel<T, V><<<grid, s->thrB, s->smemB, s->stream>>>(s->g, S, wsp<cx<T>>(s, s->off_S2), wsp<T>(s, s->off_Kh), tw, st);
}
template <typename T, int NZ> static void launch_C2(mm_sim* s, unsigned grid, cx<T>* S, twiddles<T> tw, T sc, const DevState* st)
{
    if (NZ <= 4 && s->g.xpad) {
        if (!raise_smem_limit(s, (const void*)inv_zx2_kernel<T, NZ, (NZ <= 4)>)) return;
        inv_zx2_kernel<T, NZ, (NZ <= 4)><<<grid, s->thrA, s->smemA2, s->stream>>>(s->g, S, wsp<T>(s, s->off_Hd), tw, sc, st);
        return;
    }
    if (!raise_smem_limit(s, (const void*)inv_zx2_kernel<T, NZ, false>)) return;
    inv_zx2_kernel<T, NZ, false><<<grid, s->thrA, s->smemA2, s->stream>>>(s->g, S, wsp<T>(s, s->off_Hd), tw, sc, st);
}
template <typename T, int V> static void launch_B2(mm_sim* s, unsigned grid, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    if (!raise_smem_limit(s, (const void*)y_conv2_kernel<T, V>)) return;
    y_conv2_kernel<T, V><<<grid, s->thrB, s->smemB, s->stream>>>(s->g, S, wsp<T>(s, s->off_Kc), tw, st);
}

template <typename T, int V> static void launch_B5(mm_sim* s, unsigned grid, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    if (!raise_smem_limit(s, (const void*)y_conv5_kernel<T, V>)) return;
    y_conv5_kernel<T, V><<<grid, s->thrB, s->smemB, s->stream>>>(s->g, S, wsp<T>(s, s->off_Kc), tw, st, s->tmS);
}

template <typename T> static bool b7_applies(const mm_sim* s)
{
    const Geom& g = s->g;
    if (sizeof(T) == 4 && s->b7_narrow) return g.TC == 2 && s->thrB == (g.logny >= 10 ? 256 : 128);
    return s->use_v2 && !s->no_b7 && !s->use_b3 && !s->use_b4 && g.logny >= 4 && g.logny <= 10 && g.TC == (sizeof(T) == 8 ? 2 : 4) &&
           s->thrB == (sizeof(T) == 8 ? 128 : 256) * (g.logny >= 10 ? 2 : 1);
}
template <typename T, int LOGM, bool IS3D> static void launch_B7(mm_sim* s, unsigned grid, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    if (!raise_smem_limit(s, (const void*)y_conv7_kernel<T, LOGM, IS3D>)) return;
    y_conv7_kernel<T, LOGM, IS3D><<<grid, s->thrB, s->smemB, s->stream>>>(s->g, S, wsp<T>(s, s->off_Kc), tw, ilog2(s->twN), st, s->tmS);
}
// ny = 2^4 .. 2^9 with the TMA tile of 32-byte rows: the specialised kernel; false = not covered
template <typename T> static bool try_launch_B7(mm_sim* s, unsigned grid, cx<T>* S, twiddles<T> tw, const DevState* st)
{
    const Geom& g = s->g;
    if (!s->use_tma || !b7_applies<T>(s)) return false;
    const bool d3 = g.nz > 1;
    if (sizeof(T) == 4 && s->b7_narrow && g.logny == 10) {
        if (d3) { if (raise_smem_limit(s, (const void*)y_conv7_kernel<float, 10, true, true>)) y_conv7_kernel<float, 10, true, true><<<grid, 256, s->smemB, s->stream>>>(s->g, (cx<float>*)S, (const float*)wsp<float>(s, s->off_Kc), *reinterpret_cast<twiddles<float>*>(&tw), ilog2(s->twN), st, s->tmS); }
        else { if (raise_smem_limit(s, (const void*)y_conv7_kernel<float, 10, false, true>)) y_conv7_kernel<float, 10, false, true><<<grid, 256, s->smemB, s->stream>>>(s->g, (cx<float>*)S, (const float*)wsp<float>(s, s->off_Kc), *reinterpret_cast<twiddles<float>*>(&tw), ilog2(s->twN), st, s->tmS); }
        return true;
    }
    if (sizeof(T) == 4 && s->b7_narrow) {
        if (d3) { if (raise_smem_limit(s, (const void*)y_conv7_kernel<float, 9, true, true>)) y_conv7_kernel<float, 9, true, true><<<grid, 128, s->smemB, s->stream>>>(s->g, (cx<float>*)S, (const float*)wsp<float>(s, s->off_Kc), *reinterpret_cast<twiddles<float>*>(&tw), ilog2(s->twN), st, s->tmS); }
        else { if (raise_smem_limit(s, (const void*)y_conv7_kernel<float, 9, false, true>)) y_conv7_kernel<float, 9, false, true><<<grid, 128, s->smemB, s->stream>>>(s->g, (cx<float>*)S, (const float*)wsp<float>(s, s->off_Kc), *reinterpret_cast<twiddles<float>*>(&tw), ilog2(s->twN), st, s->tmS); }
        return true;
    }
    switch (g.logny) {
#define MM_B7_CASE(L) case L: if (d3) launch_B7<T, L, true>(s, grid, S, tw, st); else launch_B7<T, L, false>(s, grid, S, tw, st); return true;
        MM_B7_CASE(4) MM_B7_CASE(5) MM_B7_CASE(6) MM_B7_CASE(7) MM_B7_CASE(8) MM_B7_CASE(9) MM_B7_CASE(10)
#undef MM_B7_CASE
        default: return false;
    }
}

// Tensor map of the spectrum S[comp][zpos][j][xpos] for pass B's box copies (TC columns x <= 256 rows).
// cuTensorMapEncodeTiled comes from the driver through the runtime's entry-point query (no -lcuda).
static int make_tmap(mm_sim* s)
{
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                 const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    const Geom& g = s->g;
    const size_t cs = 2 * esize(s);
    s->use_tma = 0;
    // measured (cfg4, B200): fp32, two CTAs per SM: TMA form 0.248 ms vs 0.254; fp64, one CTA per SM: 0.560 vs
    // 0.523 (nothing overlaps the wait for the whole tile) -> on for fp32 only; MM_TMA=0/1 overrides
    int want = s->prec == MM_F32 || b7_applies<double>(s);
    if (getenv("MM_TMA")) want = atoi(getenv("MM_TMA"));
    if (!want || !s->use_v2 || g.ny < 16) return MM_OK;
    if ((g.Lx * cs) % 16 || g.TC * cs < 16 || g.ny > 256 * 64) return MM_OK;
    EncodeFn enc = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", (void**)&enc, cudaEnableDefault, &qr) != cudaSuccess || !enc) { cudaGetLastError(); return MM_OK; }
    const cuuint64_t ew = cs / 8;      // 8-byte tensor-map elements per complex number
    cuuint64_t dims[4] = { (cuuint64_t)g.Lx * ew, (cuuint64_t)g.ny, (cuuint64_t)g.pz, 3 };
    cuuint64_t strides[3] = { (cuuint64_t)g.Lx * cs, (cuuint64_t)g.plane * cs, (cuuint64_t)g.comp * cs };
    cuuint32_t box[4] = { (cuuint32_t)(g.TC * ew), (cuuint32_t)(g.ny < 256 ? g.ny : 256), 1, 1 };
    cuuint32_t es[4] = { 1, 1, 1, 1 };
    const CUresult r = enc(&s->tmS, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, wsp<char>(s, s->off_S), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r == CUDA_SUCCESS) s->use_tma = 1;
    return MM_OK;
}

template <typename T> static int demag_passes(mm_sim* s, const T* y)
{
    const Geom& g = s->g;
    twiddles<T> tw; tw.tw = wsp<cx<T>>(s, s->off_tw); tw.twN = s->twN;
    const DevState* st = wsp<DevState>(s, s->off_st);
    cx<T>* S = wsp<cx<T>>(s, s->off_S);
    const unsigned gridA = 3u * (unsigned)(g.ny / g.G), gridB = (unsigned)(g.Lx / g.TC) * (unsigned)g.pz;
    const double P = (double)g.px * g.py * g.pz;
    const bool a2 = s->use_v2 && g.nx >= 32 && g.nz <= (sizeof(T) == 8 ? 16 : 32);
    const bool b2 = s->use_v2 && g.ny >= 16;
    prof_begin(s, 0);
    if (!a2) fwd_xz_kernel<T><<<gridA, s->thrA, s->smemA, s->stream>>>(g, y, wsp<T>(s, s->off_Ms), S, tw, st);
    else switch (g.nz) {
        case 1: launch_A2<T, 1>(s, gridA, y, S, tw, st); break;
        case 2: launch_A2<T, 2>(s, gridA, y, S, tw, st); break;
        case 4: launch_A2<T, 4>(s, gridA, y, S, tw, st); break;
        case 8: launch_A2<T, 8>(s, gridA, y, S, tw, st); break;
        case 16: launch_A2<T, 16>(s, gridA, y, S, tw, st); break;
        default: launch_A2<T, 32>(s, gridA, y, S, tw, st); break;
    }
    prof_end(s);
    prof_begin(s, 1);
    if (b2 && s->use_b4) {
        constexpr int V4 = sizeof(T) == 4 ? 2 : 1;
        if (s->clQ == 4) { if (g.TC % V4 == 0) launch_B4<T, V4, 4>(s, gridB, S, tw, st); else launch_B4<T, 1, 4>(s, gridB, S, tw, st); }
        else { if (g.TC % V4 == 0) launch_B4<T, V4, 2>(s, gridB, S, tw, st); else launch_B4<T, 1, 2>(s, gridB, S, tw, st); }
    } else if (b2 && s->use_b3) {
        if (sizeof(T) == 4 && g.TC % 2 == 0) launch_B3<T, (sizeof(T) == 4 ? 2 : 1)>(s, gridB, S, tw, st);
        else launch_B3<T, 1>(s, gridB, S, tw, st);
        S = wsp<cx<T>>(s, s->off_S2);      // pass C reads the half-tile form's output buffer
    } else if (b2 && try_launch_B7<T>(s, gridB, S, tw, st)) {
    } else if (b2 && s->use_tma) {
        if (sizeof(T) == 4 && g.TC % 2 == 0) launch_B5<T, (sizeof(T) == 4 ? 2 : 1)>(s, gridB, S, tw, st);
        else launch_B5<T, 1>(s, gridB, S, tw, st);
    } else if (!b2) y_conv_kernel<T><<<gridB, s->thrB, s->smemB, s->stream>>>(g, S, wsp<T>(s, s->off_Kh), tw, st);
    else if (sizeof(T) == 4 && g.TC % 2 == 0) launch_B2<T, (sizeof(T) == 4 ? 2 : 1)>(s, gridB, S, tw, st);
    else launch_B2<T, 1>(s, gridB, S, tw, st);
    prof_end(s);
    prof_begin(s, 2);
    if (!a2) inv_zx_kernel<T><<<gridA, s->thrA, s->smemA, s->stream>>>(g, S, wsp<T>(s, s->off_Hd), tw, (T)(1.0 / P), st);
    else switch (g.nz) {
        case 1: launch_C2<T, 1>(s, gridA, S, tw, (T)(1.0 / P), st); break;
        case 2: launch_C2<T, 2>(s, gridA, S, tw, (T)(1.0 / P), st); break;
        case 4: launch_C2<T, 4>(s, gridA, S, tw, (T)(1.0 / P), st); break;
        case 8: launch_C2<T, 8>(s, gridA, S, tw, (T)(1.0 / P), st); break;
        case 16: launch_C2<T, 16>(s, gridA, S, tw, (T)(1.0 / P), st); break;
        default: launch_C2<T, 32>(s, gridA, S, tw, (T)(1.0 / P), st); break;
    }
    prof_end(s);
    s->launches += 3;
    if (s->launch_skipped) { s->launch_skipped = false; cudaGetLastError(); return MM_ERR_CUDA; }   // s->err set where it happened
    MM_TRY(s, cudaGetLastError());
    return MM_OK;
}

// one evaluation: MODE 0 -> H, MODE 1 -> k (+ stage algebra)
template <typename T, int MODE, int S, bool NEXT, bool ERR, bool MAXK>
static void launch_stage(mm_sim* s, const LocalP<T>& lp, const T* y, const T* Hd, T* out, const StageArgs<T>& sa)
{
    // fp64: one cell per thread (148 instead of 228 registers; cfg4 stage kernel 154.3 -> 148.2 us)
    constexpr int CPT = sizeof(T) == 8 ? 1 : MM_STAGEV_CPT;
    if (s->g.nx % CPT == 0 && !s->no_stagev) {
        const unsigned blocks = (unsigned)((s->g.N / CPT + MM_STAGEV_THREADS - 1) / MM_STAGEV_THREADS);
        // general form: cell-based A / D, thermal field, Zhang-Li / Slonczewski torques, Cayley stages
        if (MODE == 2 || lp.Acell != nullptr || lp.Dcell != nullptr || lp.Hth != nullptr || lp.stt_on || lp.sl_on)
            llg_stagev_kernel<T, CPT, MODE, S, NEXT, ERR, MAXK, true><<<blocks, MM_STAGEV_THREADS, 0, s->stream>>>(s->g, lp, y, wsp<T>(s, s->off_Ms), wsp<unsigned char>(s, s->off_nbm), Hd, out, sa, wsp<DevState>(s, s->off_st));
        else if (MODE != 2)
            llg_stagev_kernel<T, CPT, MODE == 2 ? 1 : MODE, S, NEXT, ERR, MAXK, false><<<blocks, MM_STAGEV_THREADS, 0, s->stream>>>(s->g, lp, y, wsp<T>(s, s->off_Ms), wsp<unsigned char>(s, s->off_nbm), Hd, out, sa, wsp<DevState>(s, s->off_st));
        return;
    }
    const unsigned blocks = (unsigned)((s->g.N + 255) / 256);
    llg_stage_kernel<T, MODE, S, NEXT, ERR, MAXK><<<blocks, 256, 0, s->stream>>>(s->g, lp, y, wsp<T>(s, s->off_Ms), Hd, out, sa, wsp<DevState>(s, s->off_st));
}

template <typename T, int MODE> static int eval(mm_sim* s, const T* y, T* out, const StageArgs<T>& sa, int terms, bool in_step = false)
{
    const bool demag = s->demag_on && (terms & 16);
    if (demag) {
        if (!s->demag_ready) return fail(s, MM_ERR_STATE, "demag enabled but mm_init_demag not called");
        int rc = demag_passes<T>(s, y);
        if (rc) return rc;
    }
    const LocalP<T> lp = make_local<T>(s, terms, in_step);
    const T* Hd = demag ? wsp<T>(s, s->off_Hd) : (const T*)nullptr;
    prof_begin(s, 3);
    if (MODE == 2) switch (sa.s) {      // Cayley-transform RK4: d omega/dt stages (Eq. 49)
        case 0: launch_stage<T, 2, 0, true, false, true>(s, lp, y, Hd, out, sa); break;
        case 1: launch_stage<T, 2, 1, true, false, false>(s, lp, y, Hd, out, sa); break;
        case 2: launch_stage<T, 2, 2, true, false, false>(s, lp, y, Hd, out, sa); break;
        default: launch_stage<T, 2, 3, true, false, false>(s, lp, y, Hd, out, sa); break;
    }
    else if (MODE == 0) launch_stage<T, 0, 0, false, false, false>(s, lp, y, Hd, out, sa);
    else if (sa.do_err) launch_stage<T, 1, 6, false, true, false>(s, lp, y, Hd, out, sa);          // DOPRI5 stage 7
    else if (sa.ynext == nullptr) launch_stage<T, 1, 0, false, false, false>(s, lp, y, Hd, out, sa);
    else switch (sa.s) {
        case 0: launch_stage<T, 1, 0, true, false, true>(s, lp, y, Hd, out, sa); break;
        case 1: launch_stage<T, 1, 1, true, false, false>(s, lp, y, Hd, out, sa); break;
        case 2: launch_stage<T, 1, 2, true, false, false>(s, lp, y, Hd, out, sa); break;
        case 3: launch_stage<T, 1, 3, true, false, false>(s, lp, y, Hd, out, sa); break;
        case 4: launch_stage<T, 1, 4, true, false, false>(s, lp, y, Hd, out, sa); break;
        default: launch_stage<T, 1, 5, true, false, false>(s, lp, y, Hd, out, sa); break;
    }
    prof_end(s);
    s->launches++;
    MM_TRY(s, cudaGetLastError());
    return MM_OK;
}

template <typename T> static StageArgs<T> no_stage()
{
    StageArgs<T> sa;
    memset(&sa, 0, sizeof(sa));
    return sa;
}

static int set_state(mm_sim* s, double dt, double tol, double t_end, double stop, int mode, int reset)
{
    set_state_kernel<<<1, 1, 0, s->stream>>>(wsp<DevState>(s, s->off_st), dt, tol, t_end, stop, mode, reset);
    s->launches++;
    MM_TRY(s, cudaGetLastError());
    return MM_OK;
}

#define NEED_READY(s) do { NEED_WS(s); if (!(s)->Ms_set) return fail((s), MM_ERR_STATE, "Ms not set"); MM_TRY((s), cudaSetDevice((s)->device)); } while (0)

static int in_effective_field(mm_sim* s, const void* dev_m, void* dev_H)
{
    NEED_READY(s);
    if (!dev_m || !dev_H) return MM_ERR_ARG;
    int rc = set_state(s, 0, 0, 0, 0, 0, 1);
    if (rc) return rc;
    if (s->prec == MM_F64) return eval<double, 0>(s, (const double*)dev_m, (double*)dev_H, no_stage<double>(), ALL_TERMS);
    return eval<float, 0>(s, (const float*)dev_m, (float*)dev_H, no_stage<float>(), ALL_TERMS);
}

static int in_llg_rhs(mm_sim* s, const void* dev_m, void* dev_dmdt)
{
    NEED_READY(s);
    if (!dev_m || !dev_dmdt) return MM_ERR_ARG;
    int rc = set_state(s, 0, 0, 0, 0, 0, 1);
    if (rc) return rc;
    if (s->prec == MM_F64) return eval<double, 1>(s, (const double*)dev_m, (double*)dev_dmdt, no_stage<double>(), ALL_TERMS);
    return eval<float, 1>(s, (const float*)dev_m, (float*)dev_dmdt, no_stage<float>(), ALL_TERMS);
}

static int in_thermal_field(mm_sim* s, double dt, unsigned long long step, void* dev_out)
{
    NEED_READY(s);
    if (!dev_out || !(dt > 0)) return MM_ERR_ARG;
    const long N = s->g.N;
    const double V = s->dx * s->dy * s->dz;
    const double amp2 = thermal_on(s) ? 2.0 * s->alpha * KB * s->temperature / (MU0 * s->gamma * V) : 0.0;
    const unsigned blocks = (unsigned)((N + 255) / 256);
    if (s->prec == MM_F64) thermal_kernel<double><<<blocks, 256, 0, s->stream>>>(s->g, s->unx, s->uny, wsp<double>(s, s->off_Ms), amp2, s->th_seed, dt, (long long)step, wsp<DevState>(s, s->off_st), (double*)dev_out);
    else thermal_kernel<float><<<blocks, 256, 0, s->stream>>>(s->g, s->unx, s->uny, wsp<float>(s, s->off_Ms), amp2, s->th_seed, dt, (long long)step, wsp<DevState>(s, s->off_st), (float*)dev_out);
    s->launches++;
    MM_TRY(s, cudaGetLastError());
    return MM_OK;
}

// ------------------------------------------------------------------------------------------------
// Time stepping (R8).  All kernels of a step are enqueued back to back; the accept /
// reject decision and the next dt are taken on the device by ctrl_kernel.
// ------------------------------------------------------------------------------------------------
static const double DP_A[7][7] = {
    { 0 },
    { 1.0 / 5 },
    { 3.0 / 40, 9.0 / 40 },
    { 44.0 / 45, -56.0 / 15, 32.0 / 9 },
    { 19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729 },
    { 9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656 },
    { 35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84 } };
static const double DP_E[7] = { 71.0 / 57600, 0, -71.0 / 16695, 71.0 / 1920, -17253.0 / 339200, 22.0 / 525, -1.0 / 40 };
static const double RK4_A[4][4] = { { 0.5 }, { 0, 0.5 }, { 0, 0, 1.0 }, { 1.0 / 6, 1.0 / 3, 1.0 / 3, 1.0 / 6 } };

template <typename T> static int enqueue_step(mm_sim* s, T* m, int ctrl_mode)
{
    const long N = s->g.N;
    T* k[7];
    for (int i = 0; i < 7; i++) k[i] = wsp<T>(s, s->off_k[i]);
    T* yb[2] = { wsp<T>(s, s->off_y[0]), wsp<T>(s, s->off_y[1]) };
    const int nst = s->integ == MM_DOPRI5 ? 7 : 4;
    const bool thermal = thermal_on(s);
    if (thermal) {      // Eq. 42: one field per step attempt, drawn with this attempt's dt, held over its stages
        const double V = s->dx * s->dy * s->dz;
        thermal_kernel<T><<<(unsigned)((N + 255) / 256), 256, 0, s->stream>>>(s->g, s->unx, s->uny, wsp<T>(s, s->off_Ms), 2.0 * s->alpha * KB * s->temperature / (MU0 * s->gamma * V),
                                                                              s->th_seed, 0.0, -1, wsp<DevState>(s, s->off_st), wsp<T>(s, s->off_Hth));
        s->launches++;
    }
    for (int st = 0; st < nst; st++) {
        StageArgs<T> sa = no_stage<T>();
        sa.m0 = m; sa.s = st;
        {   // stage time t + c dt: row sums of the tableau
            static const double DP_C[7] = { 0.0, 1.0 / 5, 3.0 / 10, 4.0 / 5, 8.0 / 9, 1.0, 1.0 }, RK4_C[4] = { 0.0, 0.5, 0.5, 1.0 };
            sa.cstage = (T)(s->integ == MM_DOPRI5 ? DP_C[st] : RK4_C[st]);
        }
        for (int j = 0; j < st && j < 6; j++) sa.kprev[j] = k[j];
        sa.do_maxk = st == 0;
        if (s->integ == MM_DOPRI5) {
            if (st < 6) { sa.ynext = yb[st & 1]; for (int j = 0; j <= st; j++) sa.coef[j] = (T)DP_A[st + 1][j]; }
            else { sa.ynext = nullptr; sa.do_err = 1; for (int j = 0; j < 7; j++) sa.ecoef[j] = (T)DP_E[j]; }
        } else {
            // RK4 and Cayley-RK4 (k_j = d omega/dt there; omega of stage st = dt * RK4_A[st - 1] . k)
            sa.ynext = yb[st & 1];
            for (int j = 0; j <= st; j++) sa.coef[j] = (T)RK4_A[st][j];
            if (st > 0) for (int j = 0; j < st; j++) sa.wcoef[j] = (T)RK4_A[st - 1][j];
        }
        const T* y = st == 0 ? m : yb[(st - 1) & 1];
        int rc = s->integ == MM_CAYLEY_RK4 ? eval<T, 2>(s, y, k[st], sa, ALL_TERMS, true) : eval<T, 1>(s, y, k[st], sa, ALL_TERMS, true);
        if (rc) return rc;
    }
    DevState* ds = wsp<DevState>(s, s->off_st);
    ctrl_kernel<<<1, 1, 0, s->stream>>>(ds, s->prec == MM_F64, ctrl_mode, thermal ? 1 : 0, nst);
    const T* ysol = yb[1];     // DOPRI5: y_6 written at stage 5 ; RK4 / Cayley: solution written at stage 3
    accept_kernel<T><<<(unsigned)((N + 255) / 256), 256, 0, s->stream>>>(N, ds, ysol, wsp<T>(s, s->off_Ms), m, s->integ == MM_CAYLEY_RK4 ? 0 : 1);
    s->launches += 2;
    MM_TRY(s, cudaGetLastError());
    return MM_OK;
}

static int enqueue_step_eager(mm_sim* s, void* m, int ctrl_mode)
{
    return s->prec == MM_F64 ? enqueue_step<double>(s, (double*)m, ctrl_mode) : enqueue_step<float>(s, (float*)m, ctrl_mode);
}

// Everything a captured step bakes into its kernel arguments: a graph is replayed only while all of it is unchanged.
// (dt, tol, the clock, the thermal attempt counter and m itself live in device memory and are read at run time.)
static size_t step_key(const mm_sim* s, const void* m, int ctrl_mode, unsigned char* out)
{
    // `out` holds STEP_KEY_MAX bytes (the local in enqueue_step_any and StepGraph::key).  A field that would not fit is
    // not written and the returned length exceeds STEP_KEY_MAX: the caller then steps without a graph, so a key that
    // outgrows the buffer costs replay speed, never a stack overrun or a stale graph.
    size_t n = 0;
    auto put = [&](const void* p, size_t b) { if (n + b <= STEP_KEY_MAX) memcpy(out + n, p, b); n += b; };
    put(&m, sizeof(m)); put(&ctrl_mode, sizeof(int)); put(&s->ws, sizeof(void*));
    put(&s->A, sizeof(double)); put(&s->D, sizeof(double)); put(&s->Ku, sizeof(double)); put(&s->Kc, sizeof(double));
    put(s->u, sizeof(s->u)); put(s->hext, sizeof(s->hext)); put(&s->alpha, sizeof(double)); put(&s->gamma, sizeof(double));
    put(&s->dmi_kind, sizeof(int)); put(&s->integ, sizeof(int)); put(&s->demag_on, sizeof(int)); put(&s->demag_ready, sizeof(int));
    put(&s->A_cell, sizeof(int)); put(&s->D_cell, sizeof(int)); put(&s->H_cell, sizeof(int));
    put(s->stt_u, sizeof(s->stt_u)); put(&s->stt_beta, sizeof(double)); put(&s->stt_b, sizeof(double)); put(&s->stt_w, sizeof(double)); put(&s->sl_aJ, sizeof(double)); put(&s->sl_bJ, sizeof(double));
    put(s->sl_p, sizeof(s->sl_p)); put(&s->temperature, sizeof(double)); put(&s->th_seed, sizeof(s->th_seed));
    return n;
}

// One step: replayed from a captured CUDA graph when possible (SURVEY 7 hard part 5: small meshes are launch bound —
// ~30 kernels of a few microseconds each per DOPRI5 step), enqueued kernel by kernel otherwise.
static int enqueue_step_any(mm_sim* s, void* m, int ctrl_mode)
{
    if (!s->use_graph || s->prof_on) return enqueue_step_eager(s, m, ctrl_mode);
    unsigned char key[STEP_KEY_MAX];
    const size_t klen = step_key(s, m, ctrl_mode, key);
    if (klen > STEP_KEY_MAX) return enqueue_step_eager(s, m, ctrl_mode);
    mm_sim::StepGraph* e = nullptr;
    for (auto& g : s->graphs) if (g.key_len == klen && memcmp(g.key, key, klen) == 0) { e = &g; break; }
    if (!e) {      // first step with this key: run it eagerly (this also sets the kernels' shared-memory attributes)
        if (s->graphs.size() >= 8) { if (s->graphs[0].exec) cudaGraphExecDestroy(s->graphs[0].exec); s->graphs.erase(s->graphs.begin()); }
        mm_sim::StepGraph g;
        memcpy(g.key, key, klen); g.key_len = klen; g.exec = nullptr; g.launches = 0;
        s->graphs.push_back(g);
        return enqueue_step_eager(s, m, ctrl_mode);
    }
    if (!e->exec) {      // second step: capture
        if (!s->cap_stream && cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); s->use_graph = 0; return enqueue_step_eager(s, m, ctrl_mode); }
        cudaStream_t user = s->stream;
        const long l0 = s->launches;
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); s->use_graph = 0; return enqueue_step_eager(s, m, ctrl_mode); }
        s->stream = s->cap_stream;
        const int rc = enqueue_step_eager(s, m, ctrl_mode);
        s->stream = user;
        const cudaError_t ce = cudaStreamEndCapture(s->cap_stream, &graph);
        e->launches = s->launches - l0;
        s->launches = l0;
        if (rc != MM_OK || ce != cudaSuccess || !graph || cudaGraphInstantiate(&e->exec, graph, 0) != cudaSuccess) {
            cudaGetLastError();
            if (graph) cudaGraphDestroy(graph);
            e->exec = nullptr; s->use_graph = 0;
            return enqueue_step_eager(s, m, ctrl_mode);
        }
        cudaGraphDestroy(graph);
    }
    MM_TRY(s, cudaGraphLaunch(e->exec, s->stream));
    s->launches += e->launches;
    return MM_OK;
}

static int read_state(mm_sim* s, DevState* h)
{
    MM_TRY(s, cudaMemcpyAsync(h, wsp<DevState>(s, s->off_st), sizeof(DevState), cudaMemcpyDeviceToHost, s->stream));
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    s->t_host = h->t;
    return MM_OK;
}

extern "C" int mm_get_stats(mm_sim* s, long* accepted, long* rejected, long* rhs_evals)
{
    NEED_WS(s);
    MM_TRY(s, cudaSetDevice(s->device));
    DevState h;
    int rc = read_state(s, &h);
    if (rc) return rc;
    if (accepted) *accepted = (long)h.nacc;
    if (rejected) *rejected = (long)h.nrej;
    if (rhs_evals) *rhs_evals = (long)h.nrhs;
    return MM_OK;
}

// Error control and the thermal field do not go together (include/mm.h, mm_set_temperature): xi is drawn per attempt and
// scales as 1/sqrt(dt), so a controller that rejects an attempt throws a noise realisation away because it was "hard"
// and accepted steps see biased noise; Eq. 42 is written for a given dt.  Refused, not approximated.
static int refuse_adaptive_thermal(mm_sim* s, double tol)
{
    if (s->temperature > 0.0 && tol > 0.0 && s->integ == MM_DOPRI5)
        return fail(s, MM_ERR_UNSUPPORTED, "adaptive step control (tol > 0) is not available with the thermal field (T > 0): use fixed steps, tol <= 0");
    return MM_OK;
}

static int in_step(mm_sim* s, void* dev_m, double dt, double tol, int* accepted, double* err, double* dt_next, double* max_dmdt)
{
    NEED_READY(s);
    if (!dev_m || !(dt > 0)) return MM_ERR_ARG;
    if (refuse_adaptive_thermal(s, tol)) return MM_ERR_UNSUPPORTED;
    int rc = set_state(s, dt, s->integ == MM_DOPRI5 ? tol : 0.0, 0, 0, 0, 1);
    if (rc) return rc;
    if ((rc = enqueue_step_any(s, dev_m, 0))) return rc;
    if (accepted || err || dt_next || max_dmdt) {
        DevState h;
        if ((rc = read_state(s, &h))) return rc;
        if (accepted) *accepted = h.accepted;
        if (err) *err = h.err;
        if (dt_next) *dt_next = h.dt;
        if (max_dmdt) *max_dmdt = h.maxk;
        if (h.nan) return fail(s, MM_ERR_NAN, "non-finite error norm or torque");
    }
    return MM_OK;
}

static int adaptive_loop(mm_sim* s, void* dev_m, double tol, double dt0, double t_end, double stop, int mode, long max_steps, long* steps_done, double* max_dmdt)
{
    if (!dev_m || !(tol > 0) || !(dt0 > 0) || max_steps < 0) return MM_ERR_ARG;
    if (s->integ != MM_DOPRI5) return fail(s, MM_ERR_ARG, "adaptive stepping needs MM_DOPRI5");
    if (refuse_adaptive_thermal(s, tol)) return MM_ERR_UNSUPPORTED;
    int rc = set_state(s, dt0, tol, t_end, stop, mode, 1);
    if (rc) return rc;
    const long poll = 16;
    long issued = 0;
    DevState h;
    memset(&h, 0, sizeof(h));
    while (issued < max_steps) {
        const long batch = (max_steps - issued) < poll ? (max_steps - issued) : poll;
        for (long i = 0; i < batch; i++) if ((rc = enqueue_step_any(s, dev_m, mode))) return rc;
        issued += batch;
        if ((rc = read_state(s, &h))) return rc;
        if (h.done) break;
    }
    // leave the controller re-armed for later calls
    if ((rc = set_state(s, h.dt, 0, 0, 0, 0, 1))) return rc;
    if (steps_done) *steps_done = (long)h.nsteps;
    if (max_dmdt) *max_dmdt = h.maxk;
    if (h.nan) return fail(s, MM_ERR_NAN, "non-finite error norm or torque");
    return MM_OK;
}

static int in_relax(mm_sim* s, void* dev_m, double tol, double stop_dmdt, long max_steps, double dt0, long* steps_done, double* max_dmdt)
{
    NEED_READY(s);
    return adaptive_loop(s, dev_m, tol, dt0, 0.0, stop_dmdt, 1, max_steps, steps_done, max_dmdt);
}

static int in_run_until(mm_sim* s, void* dev_m, double t_end, double tol, double dt0, long max_steps, long* steps_done)
{
    NEED_READY(s);
    {   // steps enqueued without a host read-back (mm_step with NULL out-pointers) have advanced the device clock
        DevState h;
        int rc = read_state(s, &h);
        if (rc) return rc;
    }
    if (!(t_end > s->t_host)) return fail(s, MM_ERR_ARG, "t_end must be later than the current time");
    const double left = t_end - s->t_host;
    return adaptive_loop(s, dev_m, tol, dt0 < left ? dt0 : left, t_end, 0.0, 2, max_steps, steps_done, nullptr);
}

extern "C" double mm_time(mm_sim* s)
{
    if (!s || !s->ws) return 0.0;
    DevState h;
    if (read_state(s, &h)) return s->t_host;
    return h.t;
}

extern "C" int mm_set_time(mm_sim* s, double t)
{
    NEED_WS(s);
    MM_TRY(s, cudaMemcpyAsync(reinterpret_cast<char*>(wsp<DevState>(s, s->off_st)) + offsetof(DevState, t), &t, sizeof(double), cudaMemcpyHostToDevice, s->stream));
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    s->t_host = t;
    return MM_OK;
}

// ------------------------------------------------------------------------------------------------
// mm_minimize: steepest descent with Barzilai-Borwein steps.  Per iteration: demag passes,
// sd_field (field, g_k, Eq. 52 partial sums), sd_ctrl (stop decision, tau_k), sd_update (Eq. 51).  The controller
// lives on the device; the host reads it back every 16 iterations.
// ------------------------------------------------------------------------------------------------
template <typename T> static int minimize_t(mm_sim* s, T* m, double tau0, double tau_min, double tau_max, double stop, long max_steps,
                                            long* steps_done, double* max_torque, double* tau_last)
{
    const long N = s->g.N;
    MinState h;
    memset(&h, 0, sizeof(h));
    h.tau = tau0; h.tau0 = tau0; h.tau_min = tau_min; h.tau_max = tau_max; h.stop = stop; h.max_steps = max_steps;
    MinState* ms = wsp<MinState>(s, s->off_min);
    MM_TRY(s, cudaMemcpyAsync(ms, &h, sizeof(h), cudaMemcpyHostToDevice, s->stream));
    int rc = set_state(s, 0, 0, 0, 0, 0, 1);      // the demag passes look at the step controller's `done`: cleared
    if (rc) return rc;
    T* G[2] = { wsp<T>(s, s->off_k[0]), wsp<T>(s, s->off_k[1]) };
    T* sprev = wsp<T>(s, s->off_k[2]);
    T* f2 = wsp<T>(s, s->off_k[3]);
    double* part = wsp<double>(s, s->off_part);
    const bool demag = s->demag_on != 0;
    if (demag && !s->demag_ready) return fail(s, MM_ERR_STATE, "demag enabled but mm_init_demag not called");
    const LocalP<T> lp = make_local<T>(s, ALL_TERMS);
    const unsigned nblk = (unsigned)((N + 255) / 256);
    long issued = 0;
    while (issued <= max_steps) {
        const long batch = (max_steps + 1 - issued) < 16 ? (max_steps + 1 - issued) : 16;
        for (long i = 0; i < batch; i++, issued++) {
            if (demag && (rc = demag_passes<T>(s, m))) return rc;
            sd_field_kernel<T><<<nblk, 256, 0, s->stream>>>(s->g, lp, m, wsp<T>(s, s->off_Ms), demag ? wsp<T>(s, s->off_Hd) : (const T*)nullptr,
                                                            G[issued & 1], G[(issued + 1) & 1], sprev, f2, part, ms);
            sd_ctrl_kernel<<<1, 256, 0, s->stream>>>(part, (long)nblk, s->prec == MM_F64, ms);
            sd_update_kernel<T><<<nblk, 256, 0, s->stream>>>(N, m, G[issued & 1], f2, wsp<T>(s, s->off_Ms), sprev, ms);
            sd_count_kernel<<<1, 1, 0, s->stream>>>(ms);
            s->launches += 4;
            MM_TRY(s, cudaGetLastError());
        }
        MM_TRY(s, cudaMemcpyAsync(&h, ms, sizeof(h), cudaMemcpyDeviceToHost, s->stream));
        MM_TRY(s, cudaStreamSynchronize(s->stream));
        if (h.done) break;
    }
    if (steps_done) *steps_done = (long)h.iter;
    if (max_torque) *max_torque = h.maxg;
    if (tau_last) *tau_last = h.tau;
    if (h.nan) return fail(s, MM_ERR_NAN, "non-finite torque in mm_minimize");
    return MM_OK;
}

static int in_minimize(mm_sim* s, void* dev_m, double tau0, double tau_min, double tau_max, double stop_torque, long max_steps,
                           long* steps_done, double* max_torque, double* tau_last)
{
    NEED_READY(s);
    if (!dev_m || !(tau0 > 0) || !(tau_min > 0) || !(tau_max >= tau_min) || max_steps < 0) return MM_ERR_ARG;
    return s->prec == MM_F64 ? minimize_t<double>(s, (double*)dev_m, tau0, tau_min, tau_max, stop_torque, max_steps, steps_done, max_torque, tau_last)
                             : minimize_t<float>(s, (float*)dev_m, tau0, tau_min, tau_max, stop_torque, max_steps, steps_done, max_torque, tau_last);
}

// ------------------------------------------------------------------------------------------------
// Host-buffer entry points (end-to-end path: H2D, compute, D2H inside the call)
// ------------------------------------------------------------------------------------------------
static int in_run_host(mm_sim* s, void* host_m, int nsteps, double dt, double tol)
{
    NEED_READY(s);
    if (!host_m || nsteps < 0 || !(dt > 0)) return MM_ERR_ARG;
    if (refuse_adaptive_thermal(s, tol)) return MM_ERR_UNSUPPORTED;
    const size_t bytes = 3 * (size_t)s->g.N * esize(s);
    // m lives in the workspace's own staging slot for the duration of the call
    void* dm = wsp<char>(s, s->off_mh);
    MM_TRY(s, cudaMemcpyAsync(dm, host_m, bytes, cudaMemcpyHostToDevice, s->stream));
    int rc = set_state(s, dt, s->integ == MM_DOPRI5 ? tol : 0.0, 0, 0, 0, 1);
    for (int i = 0; i < nsteps && !rc; i++) rc = enqueue_step_any(s, dm, 0);
    if (!rc) {
        cudaError_t e = cudaMemcpyAsync(host_m, dm, bytes, cudaMemcpyDeviceToHost, s->stream);
        if (e != cudaSuccess) { s->err = cudaGetErrorString(e); rc = MM_ERR_CUDA; }
    }
    DevState h;
    int rc2 = read_state(s, &h);
    return rc ? rc : rc2;
}

static int in_llg_rhs_host(mm_sim* s, const void* host_m, void* host_dmdt)
{
    NEED_READY(s);
    if (!host_m || !host_dmdt) return MM_ERR_ARG;
    const size_t bytes = 3 * (size_t)s->g.N * esize(s);
    void* dm = wsp<char>(s, s->off_y[0]);
    void* dk = wsp<char>(s, s->off_k[0]);
    MM_TRY(s, cudaMemcpyAsync(dm, host_m, bytes, cudaMemcpyHostToDevice, s->stream));
    int rc = in_llg_rhs(s, dm, dk);
    if (rc) return rc;
    MM_TRY(s, cudaMemcpyAsync(host_dmdt, dk, bytes, cudaMemcpyDeviceToHost, s->stream));
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    return MM_OK;
}

// ------------------------------------------------------------------------------------------------
// Diagnostics
// ------------------------------------------------------------------------------------------------
template <typename T> static int reduce_dot(mm_sim* s, const T* a, const T* b, int mode, double out4[4])
{
    const int blocks = 1024;
    double* part = wsp<double>(s, s->off_part);
    dot_kernel<T><<<blocks, 256, 0, s->stream>>>(s->g.N, a, b, wsp<T>(s, s->off_Ms), mode, part);
    s->launches++;
    MM_TRY(s, cudaGetLastError());
    std::vector<double> h(4 * blocks);
    MM_TRY(s, cudaMemcpyAsync(h.data(), part, h.size() * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    for (int c = 0; c < 4; c++) { out4[c] = 0; for (int b2 = 0; b2 < blocks; b2++) out4[c] += h[4 * b2 + c]; }
    return MM_OK;
}

static int in_average_m(mm_sim* s, const void* dev_m, double out3[3])
{
    NEED_READY(s);
    if (!dev_m || !out3) return MM_ERR_ARG;
    double r[4];
    int rc = s->prec == MM_F64 ? reduce_dot<double>(s, (const double*)dev_m, (const double*)dev_m, 1, r)
                               : reduce_dot<float>(s, (const float*)dev_m, (const float*)dev_m, 1, r);
    if (rc) return rc;
    for (int c = 0; c < 3; c++) out3[c] = r[3] > 0 ? r[c] / r[3] : 0.0;
    return MM_OK;
}

template <typename T> static int energy_t(mm_sim* s, const T* m, double* E_total, double E_terms[5])
{
    // quadratic terms carry 1/2, the quartic cubic-anisotropy term 1/4 (Euler's theorem: m.H = -4 w / (mu0 Ms)), the
    // linear Zeeman term 1; cubic anisotropy is reported inside the anisotropy slot
    static const int bits[6] = { 16, 1, 2, 4, 8, 32 };
    static const double w[6] = { 0.5, 0.5, 0.5, 0.5, 1.0, 0.25 };
    static const int slot[6] = { 0, 1, 2, 3, 4, 3 };
    T* H = wsp<T>(s, s->off_k[6]);
    const double V = s->dx * s->dy * s->dz;
    double tot = 0;
    int rc = set_state(s, 0, 0, 0, 0, 0, 1);
    if (rc) return rc;
    if (E_terms) for (int t = 0; t < 5; t++) E_terms[t] = 0.0;
    for (int t = 0; t < 6; t++) {
        if (t == 5 && s->Kc == 0.0) continue;
        if ((rc = eval<T, 0>(s, m, H, no_stage<T>(), bits[t]))) return rc;
        double r[4];
        if ((rc = reduce_dot<T>(s, m, H, 0, r))) return rc;
        const double e = -MU0 * V * w[t] * r[0];
        if (E_terms) E_terms[slot[t]] += e;
        tot += e;
    }
    if (E_total) *E_total = tot;
    return MM_OK;
}

static int in_energy(mm_sim* s, const void* dev_m, double* E_total, double E_terms[5])
{
    NEED_READY(s);
    if (!dev_m) return MM_ERR_ARG;
    return s->prec == MM_F64 ? energy_t<double>(s, (const double*)dev_m, E_total, E_terms) : energy_t<float>(s, (const float*)dev_m, E_total, E_terms);
}

// ------------------------------------------------------------------------------------------------
// The ABI entry points that take cell arrays.  A mesh whose sizes are powers of two goes straight to the inner
// functions above.  Any other mesh is EMBEDDED (SURVEY 8(f)4 "non-power-of-two meshes"): the caller's nx x ny x nz
// arrays are packed into / unpacked from the padded 2^k mesh whose extra cells are vacuum (Ms = 0: no field, no
// torque, absent as neighbours — exactly the free boundary of R4), and the demag tensor depends on offsets only, so
// every result at the caller's cells is the one of the caller's mesh.
// ------------------------------------------------------------------------------------------------
namespace mm {
// dir 0: user -> inner (zero outside the caller's mesh); dir 1: inner -> user.  One thread per inner cell.
template <typename T>
__global__ void __launch_bounds__(256) embed_kernel(Geom g, int unx, int uny, int unz, int ncomp, const T* __restrict__ src, T* __restrict__ dst, int dir)
{
    const long q = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= g.N) return;
    const int i = (int)(q & (g.nx - 1)), j = (int)((q >> g.lognx) & (g.ny - 1)), k = (int)(q >> (g.lognx + g.logny));
    const bool inside = i < unx && j < uny && k < unz;
    const long uN = (long)unx * uny * unz, uq = i + (long)unx * (j + (long)uny * k);
    for (int c = 0; c < ncomp; c++) {
        if (dir == 0) dst[c * g.N + q] = inside ? src[c * uN + uq] : (T)0;
        else if (inside) dst[c * uN + uq] = src[c * g.N + q];
    }
}
}  // namespace mm

template <typename T> static int embed_t(mm_sim* s, const void* src, void* dst, int ncomp, int dir)
{
    embed_kernel<T><<<(unsigned)((s->g.N + 255) / 256), 256, 0, s->stream>>>(s->g, s->unx, s->uny, s->unz, ncomp, (const T*)src, (T*)dst, dir);
    s->launches++;
    MM_TRY(s, cudaGetLastError());
    return MM_OK;
}
static int embed_in(mm_sim* s, const void* user, void* inner, int ncomp) { return s->prec == MM_F64 ? embed_t<double>(s, user, inner, ncomp, 0) : embed_t<float>(s, user, inner, ncomp, 0); }
static int embed_out(mm_sim* s, const void* inner, void* user, int ncomp) { return s->prec == MM_F64 ? embed_t<double>(s, inner, user, ncomp, 1) : embed_t<float>(s, inner, user, ncomp, 1); }
static void* slot_in(mm_sim* s) { return wsp<char>(s, s->off_ei); }
static void* slot_out(mm_sim* s) { return wsp<char>(s, s->off_eo); }
#define MM_EMB_CHECK(s, p) do { NEED_WS(s); if (!(p)) return MM_ERR_ARG; MM_TRY((s), cudaSetDevice((s)->device)); } while (0)

extern "C" int mm_set_Ms_uniform(mm_sim* s, double Ms)
{
    if (!s || !s->embed) return in_set_Ms_uniform(s, Ms);
    // uniform inside the caller's mesh, vacuum in the padding: fill a caller-shaped array and pack it
    NEED_WS(s);
    if (!(Ms >= 0)) return fail(s, MM_ERR_ARG, "Ms must be >= 0");
    MM_TRY(s, cudaSetDevice(s->device));
    const int blocks = (int)((s->uN + 255) / 256);
    if (s->prec == MM_F64) fill_kernel<double><<<blocks, 256, 0, s->stream>>>(s->uN, (double*)slot_out(s), Ms);
    else fill_kernel<float><<<blocks, 256, 0, s->stream>>>(s->uN, (float*)slot_out(s), (float)Ms);
    s->launches++;
    int rc = embed_in(s, slot_out(s), slot_in(s), 1);
    return rc ? rc : in_set_Ms(s, slot_in(s));
}
extern "C" int mm_set_Ms(mm_sim* s, const void* dev_Ms)
{
    if (!s || !s->embed) return in_set_Ms(s, dev_Ms);
    MM_EMB_CHECK(s, dev_Ms);
    int rc = embed_in(s, dev_Ms, slot_in(s), 1);
    return rc ? rc : in_set_Ms(s, slot_in(s));
}
extern "C" int mm_set_A_cell(mm_sim* s, const void* dev_A)
{
    if (!s || !s->embed || !dev_A) return in_set_A_cell(s, dev_A);
    MM_EMB_CHECK(s, dev_A);
    int rc = embed_in(s, dev_A, slot_in(s), 1);
    return rc ? rc : in_set_A_cell(s, slot_in(s));
}
extern "C" int mm_set_D_cell(mm_sim* s, const void* dev_D, mm_dmi_kind kind)
{
    if (!s || !s->embed || !dev_D) return in_set_D_cell(s, dev_D, kind);
    MM_EMB_CHECK(s, dev_D);
    int rc = embed_in(s, dev_D, slot_in(s), 1);
    return rc ? rc : in_set_D_cell(s, slot_in(s), kind);
}
extern "C" int mm_set_H_ext_cell(mm_sim* s, const void* dev_H)
{
    if (!s || !s->embed || !dev_H) return in_set_H_ext_cell(s, dev_H);
    MM_EMB_CHECK(s, dev_H);
    int rc = embed_in(s, dev_H, slot_in(s), 3);
    return rc ? rc : in_set_H_ext_cell(s, slot_in(s));
}
extern "C" int mm_get_demag_kernel(mm_sim* s, int comp, void* dev_out)
{
    if (!s || !s->embed) return in_get_demag_kernel(s, comp, dev_out);
    MM_EMB_CHECK(s, dev_out);
    // N doubles of the inner mesh fit the 3N-real slot in either precision (8 N <= 12 N bytes)
    int rc = in_get_demag_kernel(s, comp, slot_in(s));
    if (rc) return rc;
    rc = embed_t<double>(s, slot_in(s), dev_out, 1, 1);
    if (rc) return rc;
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    return MM_OK;
}
extern "C" int mm_effective_field(mm_sim* s, const void* dev_m, void* dev_H)
{
    if (!s || !s->embed) return in_effective_field(s, dev_m, dev_H);
    MM_EMB_CHECK(s, dev_m && dev_H);
    int rc = embed_in(s, dev_m, slot_in(s), 3);
    if (!rc) rc = in_effective_field(s, slot_in(s), slot_out(s));
    return rc ? rc : embed_out(s, slot_out(s), dev_H, 3);
}
extern "C" int mm_llg_rhs(mm_sim* s, const void* dev_m, void* dev_dmdt)
{
    if (!s || !s->embed) return in_llg_rhs(s, dev_m, dev_dmdt);
    MM_EMB_CHECK(s, dev_m && dev_dmdt);
    int rc = embed_in(s, dev_m, slot_in(s), 3);
    if (!rc) rc = in_llg_rhs(s, slot_in(s), slot_out(s));
    return rc ? rc : embed_out(s, slot_out(s), dev_dmdt, 3);
}
extern "C" int mm_thermal_field(mm_sim* s, double dt, unsigned long long step, void* dev_out)
{
    if (!s || !s->embed) return in_thermal_field(s, dt, step, dev_out);
    MM_EMB_CHECK(s, dev_out);
    int rc = in_thermal_field(s, dt, step, slot_out(s));
    return rc ? rc : embed_out(s, slot_out(s), dev_out, 3);
}
// in-place integrators: pack m, run on the inner copy, unpack (stream-ordered; the inner call decides about syncing,
// so the unpack is enqueued BEFORE a call that may read back would return — hence pack / unpack around an async core)
extern "C" int mm_step(mm_sim* s, void* dev_m, double dt, double tol, int* accepted, double* err, double* dt_next, double* max_dmdt)
{
    if (!s || !s->embed) return in_step(s, dev_m, dt, tol, accepted, err, dt_next, max_dmdt);
    MM_EMB_CHECK(s, dev_m);
    int rc = embed_in(s, dev_m, slot_in(s), 3);
    if (!rc) rc = in_step(s, slot_in(s), dt, tol, nullptr, nullptr, nullptr, nullptr);
    if (!rc) rc = embed_out(s, slot_in(s), dev_m, 3);
    if (rc) return rc;
    if (accepted || err || dt_next || max_dmdt) {
        DevState h;
        if ((rc = read_state(s, &h))) return rc;
        if (accepted) *accepted = h.accepted;
        if (err) *err = h.err;
        if (dt_next) *dt_next = h.dt;
        if (max_dmdt) *max_dmdt = h.maxk;
        if (h.nan) return fail(s, MM_ERR_NAN, "non-finite error norm or torque");
    }
    return MM_OK;
}
extern "C" int mm_relax(mm_sim* s, void* dev_m, double tol, double stop_dmdt, long max_steps, double dt0, long* steps_done, double* max_dmdt)
{
    if (!s || !s->embed) return in_relax(s, dev_m, tol, stop_dmdt, max_steps, dt0, steps_done, max_dmdt);
    MM_EMB_CHECK(s, dev_m);
    int rc = embed_in(s, dev_m, slot_in(s), 3);
    if (!rc) rc = in_relax(s, slot_in(s), tol, stop_dmdt, max_steps, dt0, steps_done, max_dmdt);
    const int rc2 = embed_out(s, slot_in(s), dev_m, 3);
    return rc ? rc : rc2;
}
extern "C" int mm_run_until(mm_sim* s, void* dev_m, double t_end, double tol, double dt0, long max_steps, long* steps_done)
{
    if (!s || !s->embed) return in_run_until(s, dev_m, t_end, tol, dt0, max_steps, steps_done);
    MM_EMB_CHECK(s, dev_m);
    int rc = embed_in(s, dev_m, slot_in(s), 3);
    if (!rc) rc = in_run_until(s, slot_in(s), t_end, tol, dt0, max_steps, steps_done);
    const int rc2 = embed_out(s, slot_in(s), dev_m, 3);
    return rc ? rc : rc2;
}
extern "C" int mm_minimize(mm_sim* s, void* dev_m, double tau0, double tau_min, double tau_max, double stop_torque, long max_steps,
                           long* steps_done, double* max_torque, double* tau_last)
{
    if (!s || !s->embed) return in_minimize(s, dev_m, tau0, tau_min, tau_max, stop_torque, max_steps, steps_done, max_torque, tau_last);
    MM_EMB_CHECK(s, dev_m);
    int rc = embed_in(s, dev_m, slot_in(s), 3);
    if (!rc) rc = in_minimize(s, slot_in(s), tau0, tau_min, tau_max, stop_torque, max_steps, steps_done, max_torque, tau_last);
    const int rc2 = embed_out(s, slot_in(s), dev_m, 3);
    return rc ? rc : rc2;
}
extern "C" int mm_run_host(mm_sim* s, void* host_m, int nsteps, double dt, double tol)
{
    if (!s || !s->embed) return in_run_host(s, host_m, nsteps, dt, tol);
    MM_EMB_CHECK(s, host_m);
    if (!s->Ms_set) return fail(s, MM_ERR_STATE, "Ms not set");
    if (nsteps < 0 || !(dt > 0)) return MM_ERR_ARG;
    const size_t bytes = 3 * (size_t)s->uN * esize(s);
    MM_TRY(s, cudaMemcpyAsync(slot_out(s), host_m, bytes, cudaMemcpyHostToDevice, s->stream));
    int rc = embed_in(s, slot_out(s), slot_in(s), 3);
    if (!rc) rc = set_state(s, dt, s->integ == MM_DOPRI5 ? tol : 0.0, 0, 0, 0, 1);
    for (int i = 0; i < nsteps && !rc; i++) rc = enqueue_step_any(s, slot_in(s), 0);
    if (!rc) rc = embed_out(s, slot_in(s), slot_out(s), 3);
    if (!rc) {
        cudaError_t e = cudaMemcpyAsync(host_m, slot_out(s), bytes, cudaMemcpyDeviceToHost, s->stream);
        if (e != cudaSuccess) { s->err = cudaGetErrorString(e); rc = MM_ERR_CUDA; }
    }
    DevState h;
    const int rc2 = read_state(s, &h);
    return rc ? rc : rc2;
}
extern "C" int mm_llg_rhs_host(mm_sim* s, const void* host_m, void* host_dmdt)
{
    if (!s || !s->embed) return in_llg_rhs_host(s, host_m, host_dmdt);
    MM_EMB_CHECK(s, host_m && host_dmdt);
    const size_t bytes = 3 * (size_t)s->uN * esize(s);
    MM_TRY(s, cudaMemcpyAsync(slot_out(s), host_m, bytes, cudaMemcpyHostToDevice, s->stream));
    int rc = embed_in(s, slot_out(s), slot_in(s), 3);
    if (!rc) rc = in_llg_rhs(s, slot_in(s), slot_out(s));
    if (!rc) rc = embed_out(s, slot_out(s), slot_in(s), 3);      // caller layout, staged in the input slot
    if (rc) return rc;
    MM_TRY(s, cudaMemcpyAsync(host_dmdt, slot_in(s), bytes, cudaMemcpyDeviceToHost, s->stream));
    MM_TRY(s, cudaStreamSynchronize(s->stream));
    return MM_OK;
}
extern "C" int mm_average_m(mm_sim* s, const void* dev_m, double out3[3])
{
    if (!s || !s->embed) return in_average_m(s, dev_m, out3);
    MM_EMB_CHECK(s, dev_m);
    int rc = embed_in(s, dev_m, slot_in(s), 3);
    return rc ? rc : in_average_m(s, slot_in(s), out3);
}
extern "C" int mm_energy(mm_sim* s, const void* dev_m, double* E_total, double E_terms[5])
{
    if (!s || !s->embed) return in_energy(s, dev_m, E_total, E_terms);
    MM_EMB_CHECK(s, dev_m);
    int rc = embed_in(s, dev_m, slot_in(s), 3);
    return rc ? rc : in_energy(s, slot_in(s), E_total, E_terms);
}
