// mm_noalloc.cu — mm_average_m_static: the mean magnetisation <m> without any memory of the caller's or the
// allocator's beyond the inputs and the 3-double output.
//
// Who this is for.  Every other compute call of libmm.so works inside a workspace of hundreds of megabytes that the
// caller allocates and hands over with mm_set_workspace; mm_average_m, for one, writes its per-block partial sums
// there.  Some users of the library have no way to produce such a buffer at the moment they want <m>:
//   * a monitoring or logging hook that runs inside a host application whose memory pool has already claimed the
//     whole of HBM — a raw cudaMalloc from the hook fails, and the hook has no access to the pool;
//   * code in the middle of a time-critical loop, where cudaMalloc / cudaFree would make every stream of the
//     device wait (both synchronise the device) and the jitter is not acceptable;
//   * a plug-in that is only ever handed the two arrays (m and Ms) and a stream, with no handle, no workspace and
//     no permission to create either.
// For them the partial sums live in the file-scope array below, which is part of the library's image: the driver
// places it when the library is loaded on a device and it stays there until the process exits (256 B + 512 KiB on
// every GPU that loads libmm.so, whether or not this call is ever made).  The call itself allocates nothing, on
// the host or on the device, and frees nothing.
//
// What the fixed array costs the caller:
//   * a size limit: at most MM_STATIC_MAX_CELLS cells (one partial-sum slot per 4096 cells); larger arrays are
//     refused with MM_ERR_UNSUPPORTED and a message, never truncated;
//   * one array per device for all callers: two calls whose kernels can be on the GPU at the same time (different
//     streams, or different host threads on different streams) write the same slots and the same ticket, and both
//     results are then undefined.  Calls on one stream are ordered by the stream and are safe;
//   * the array keeps what the previous call left in it.  Only the ticket (the count of finished blocks) has to
//     start at zero; it is cleared on the caller's stream before every launch.  The partial-sum slots need no
//     clearing: each launch overwrites every slot it later reads.
//
// The first call on a device looks up the device address of the array (cudaGetSymbolAddress), which makes the
// driver load this library's device code on that device if nothing has yet.  That is a one-off set-up cost with
// driver-side effects of its own, so make the first call on each device early, outside any stream capture and
// outside the time-critical part of the program.  Later calls only enqueue a 256-byte memset and one kernel.
#include <cuda_runtime.h>
#include <stdio.h>

#include <atomic>

#include "../../include/mm.h"

namespace {

constexpr int NA_THREADS = 256;                 // threads per block
constexpr int NA_CELLS_PER_THREAD = 16;
constexpr long NA_CELLS_PER_BLOCK = (long)NA_THREADS * NA_CELLS_PER_THREAD;          // 4096
constexpr long NA_MAX_BLOCKS = MM_STATIC_MAX_CELLS / NA_CELLS_PER_BLOCK;              // 16384
constexpr int NA_HEADER = 32;                   // doubles: a 256-byte header, its first word is the ticket
constexpr int NA_MAX_DEVICES = 64;
static_assert(MM_STATIC_MAX_CELLS % NA_CELLS_PER_BLOCK == 0, "limit must be a whole number of blocks");

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress — it is not a device address and
// must never be passed to a kernel; device_scratch() below turns it into one, per device.
static __device__ __align__(256) double mm_static_scratch[NA_HEADER + 4 * NA_MAX_BLOCKS];

thread_local char g_err[256] = "";

int fail(int code, const char* fmt, long a = 0, long b = 0)
{
    snprintf(g_err, sizeof g_err, fmt, a, b);
    return code;
}

// Device address of the scratch array on `device`, which must be the current device.  Looked up once per device.
// Two host threads racing here look up the same value and store it twice; an atomic slot is all that is needed.
std::atomic<double*> g_scratch_ptr[NA_MAX_DEVICES];

int device_scratch(int device, double** out)
{
    double* p = g_scratch_ptr[device].load(std::memory_order_acquire);
    if (!p) {
        cudaError_t e = cudaGetSymbolAddress((void**)&p, mm_static_scratch);
        if (e != cudaSuccess || !p) {
            snprintf(g_err, sizeof g_err, "mm_average_m_static: cudaGetSymbolAddress on device %d: %s", device, cudaGetErrorString(e));
            return MM_ERR_CUDA;
        }
        g_scratch_ptr[device].store(p, std::memory_order_release);
    }
    *out = p;
    return MM_OK;
}

// Block b sums m_x, m_y, m_z and the cell count over the cells [4096 b, 4096 (b+1)) with Ms != 0, in fp64, and
// stores the four numbers in its slot of `scratch`.  The block that draws the last ticket then adds the slots in a
// fixed order (slot s goes to thread s mod 256, then the same tree as above), so the result does not depend on
// which block finishes last, and writes the three means (0 if no cell has Ms != 0) to out3.
template <typename T>
__global__ void __launch_bounds__(NA_THREADS) average_m_static_kernel(long N, const T* __restrict__ m, const T* __restrict__ Ms,
                                                                      double* scratch, double* __restrict__ out3)
{
    __shared__ double red[4][NA_THREADS];
    __shared__ bool last;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    double* part = scratch + NA_HEADER;
    const int t = threadIdx.x;

    double v[4] = { 0, 0, 0, 0 };
    const long base = (long)blockIdx.x * NA_CELLS_PER_BLOCK;
#pragma unroll 4
    for (int i = 0; i < NA_CELLS_PER_THREAD; i++) {
        const long q = base + t + (long)i * NA_THREADS;
        if (q < N && (double)Ms[q] != 0.0) {
            v[0] += (double)m[q]; v[1] += (double)m[N + q]; v[2] += (double)m[2 * N + q]; v[3] += 1.0;
        }
    }
    for (int c = 0; c < 4; c++) red[c][t] = v[c];
    __syncthreads();
    for (int o = NA_THREADS / 2; o > 0; o >>= 1) {
        if (t < o) for (int c = 0; c < 4; c++) red[c][t] += red[c][t + o];
        __syncthreads();
    }
    if (t == 0) {
        for (int c = 0; c < 4; c++) part[4 * (long)blockIdx.x + c] = red[c][0];
        __threadfence();                                   // the slot is visible before the ticket is drawn
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();                                       // every other block's slot is visible to this block

    for (int c = 0; c < 4; c++) v[c] = 0;
    for (unsigned int b = t; b < gridDim.x; b += NA_THREADS)
        for (int c = 0; c < 4; c++) v[c] += __ldcg(part + 4 * (long)b + c);
    for (int c = 0; c < 4; c++) red[c][t] = v[c];
    __syncthreads();
    for (int o = NA_THREADS / 2; o > 0; o >>= 1) {
        if (t < o) for (int c = 0; c < 4; c++) red[c][t] += red[c][t + o];
        __syncthreads();
    }
    if (t < 3) out3[t] = red[3][0] > 0 ? red[t][0] / red[3][0] : 0.0;
}

}  // namespace

extern "C" const char* mm_static_last_error(void) { return g_err; }

extern "C" int mm_average_m_static(int device, void* cuda_stream, mm_prec prec, long ncells, const void* dev_m, const void* dev_Ms,
                                   double* dev_out3)
{
    // everything that can be refused without touching the GPU is refused first
    if (!dev_m || !dev_Ms || !dev_out3) return fail(MM_ERR_ARG, "mm_average_m_static: NULL pointer");
    if (prec != MM_F32 && prec != MM_F64) return fail(MM_ERR_ARG, "mm_average_m_static: precision must be MM_F32 or MM_F64");
    if (ncells < 1) return fail(MM_ERR_ARG, "mm_average_m_static: ncells = %ld, must be >= 1", ncells);
    if (ncells > MM_STATIC_MAX_CELLS)
        return fail(MM_ERR_UNSUPPORTED, "mm_average_m_static: %ld cells, but the library's built-in scratch array holds partial sums for "
                                        "at most %ld (MM_STATIC_MAX_CELLS); use mm_average_m with a workspace for larger meshes",
                    ncells, (long)MM_STATIC_MAX_CELLS);
    if (device < 0 || device >= NA_MAX_DEVICES) return fail(MM_ERR_ARG, "mm_average_m_static: device %ld outside 0..%ld", device, NA_MAX_DEVICES - 1);

    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) { snprintf(g_err, sizeof g_err, "mm_average_m_static: cudaSetDevice(%d): %s", device, cudaGetErrorString(e)); return MM_ERR_CUDA; }
    double* scratch = nullptr;
    int rc = device_scratch(device, &scratch);
    if (rc) return rc;

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const unsigned int blocks = (unsigned int)((ncells + NA_CELLS_PER_BLOCK - 1) / NA_CELLS_PER_BLOCK);
    // the ticket must start at zero whatever the previous call (finished, failed or aborted) left behind
    e = cudaMemsetAsync(scratch, 0, NA_HEADER * sizeof(double), stream);
    if (e == cudaSuccess) {
        if (prec == MM_F64) average_m_static_kernel<double><<<blocks, NA_THREADS, 0, stream>>>(ncells, (const double*)dev_m, (const double*)dev_Ms, scratch, dev_out3);
        else                average_m_static_kernel<float><<<blocks, NA_THREADS, 0, stream>>>(ncells, (const float*)dev_m, (const float*)dev_Ms, scratch, dev_out3);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) { snprintf(g_err, sizeof g_err, "mm_average_m_static: launch: %s", cudaGetErrorString(e)); return MM_ERR_CUDA; }
    g_err[0] = 0;
    return MM_OK;
}
