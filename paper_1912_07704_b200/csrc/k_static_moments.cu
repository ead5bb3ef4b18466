/*
 * k_static_moments.cu — aa_row_moments_static: the per-row checksums of K5 (sum_t D[i][t] and sum_t t*D[i][t], the
 * all-rows check of DESIGN.md "Verification") for callers that must not allocate device memory.
 *
 * Who that is. aa_get_row_moments needs a strategy: its partial sums live in the strategy's arena, and a strategy costs a
 * cudaMalloc at set-up (or an arena the caller has to find room for). Two kinds of caller cannot pay that:
 *   - a back-end that divided the GPU's memory up front (one arena lent to this library, the rest to the capture ring and
 *     to other stages): a later cudaMalloc may simply fail there, and it may not be allowed to succeed either, because the
 *     memory budget is a contract between stages;
 *   - a monitoring thread that checksums rows of D while the streaming loop runs: cudaMalloc and cudaFree synchronise the
 *     WHOLE device, so one allocation stalls the H2D prefetch and the dedispersion kernels of every stream for its duration.
 * This entry point therefore calls no cudaMalloc, no cudaFree and no library routine that allocates. Its only working
 * memory is the file-scope array below, which is part of the library image: every GPU on which this library's kernels are
 * loaded holds its own 256 KiB copy from the moment the module is loaded until the process exits, used or not.
 *
 * Kernel. k_row_moments (k_misc.cu) gives a row to ONE CTA and stores the two sums. A caller outside the pipeline typically
 * checks a few long rows, which leaves most SMs idle, so this variant cuts every row into slices, one CTA per (slice, row),
 * and each CTA adds its partial sums into the row's two scratch words with 64-bit atomics. Integer addition modulo 2^64 is
 * associative and commutative, so the result equals k_row_moments' bit for bit whatever the slicing or arrival order. The
 * scratch words therefore have to START AT ZERO: a small kernel clears the words the call is about to use, on the caller's stream
 * ahead of the summing kernel, every call (the array keeps whatever the previous call left).
 */
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "aa_internal.h"

/* The scratch, at file scope: [0, MAX_ROWS) holds sum_t D of each row, [MAX_ROWS, 2 MAX_ROWS) holds sum_t t*D.
 * 2 x 16384 x 8 B = 256 KiB per GPU. In HOST code this name is only a handle to give to cudaGetSymbolAddress, not a device
 * address: a kernel handed `g_moment_scratch` itself would fault (or scribble on host memory where the GPU can reach it).
 * Host code below passes the address that cudaGetSymbolAddress returned for the current device. */
static __device__ __align__(256) unsigned long long g_moment_scratch[2 * AA_STATIC_MOMENTS_MAX_ROWS];

namespace {

typedef unsigned long long u64;

constexpr int kMaxRows = AA_STATIC_MOMENTS_MAX_ROWS;      /* rows per call; sizes the scratch array */
constexpr int kThreads = 256;
constexpr long long kSliceMin = 16384;                    /* samples per CTA before a row is cut further */
constexpr int kMaxSlices = 64;
constexpr int kMaxDevices = 64;

/* Device address of g_moment_scratch on each device, filled on the first call made with that device current. */
std::mutex g_setup_mutex;
u64* g_scratch_on_device[kMaxDevices];

__global__ void __launch_bounds__(kThreads)
k_row_moments_sliced(const int32_t* __restrict__ D, long long pitch, long long nt, long long slice_len, u64* __restrict__ scratch) {
    __shared__ long long red[2 * (kThreads / 32)];
    const int32_t* row = D + (size_t)blockIdx.y * (size_t)pitch;
    const long long t0 = (long long)blockIdx.x * slice_len;
    const long long t1 = t0 + slice_len < nt ? t0 + slice_len : nt;
    long long a = 0, b = 0;
    for (long long t = t0 + threadIdx.x; t < t1; t += kThreads) { const long long v = row[t]; a += v; b += v * t; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o); }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { red[warp * 2] = a; red[warp * 2 + 1] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long sa = 0, sb = 0;
        for (int w = 0; w < kThreads / 32; ++w) { sa += red[w * 2]; sb += red[w * 2 + 1]; }
        /* two's complement: adding the bit patterns as unsigned is the signed sum modulo 2^64 */
        atomicAdd(scratch + blockIdx.y, (u64)sa);
        atomicAdd(scratch + kMaxRows + blockIdx.y, (u64)sb);
    }
}

/* Device code may name the array directly (only host code needs the looked-up address): zero the words of rows [0, nrows). */
__global__ void __launch_bounds__(kThreads) k_clear_moment_scratch(int nrows) {
    const int i = blockIdx.x * kThreads + threadIdx.x;
    if (i < nrows) { g_moment_scratch[i] = 0ull; g_moment_scratch[kMaxRows + i] = 0ull; }
}

/* Once per device, with that device current: ask the runtime where g_moment_scratch lives on it. */
aa_status scratch_of_current_device(u64** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return aa::cuda_fail(e, "aa_row_moments_static: cudaGetDevice");
    if (dev < 0 || dev >= kMaxDevices) {
        aa::set_error("aa_row_moments_static: device ordinal %d is beyond the %d devices this entry point keeps an address for", dev, kMaxDevices);
        return AA_ERR_INVALID_ARG;
    }
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_on_device[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_moment_scratch);
        if (e != cudaSuccess || !p) return aa::cuda_fail(e != cudaSuccess ? e : cudaErrorInvalidSymbol, "aa_row_moments_static: cudaGetSymbolAddress(g_moment_scratch)");
        g_scratch_on_device[dev] = static_cast<u64*>(p);
    }
    *out = g_scratch_on_device[dev];
    return AA_OK;
}

}  // namespace

static_assert(AA_STATIC_MOMENTS_MAX_ROWS == 16384, "include/aa.h states the limit in words as well: keep the two in step");

extern "C" aa_status aa_row_moments_static(const int32_t* device_D, int64_t row_pitch, int64_t nt, int32_t nrows,
                                           int64_t* host_sum_d, int64_t* host_sum_td, void* stream) {
    if (nrows < 0 || nrows > kMaxRows) {
        aa::set_error("aa_row_moments_static: nrows = %d, but one call takes at most AA_STATIC_MOMENTS_MAX_ROWS = %d rows (the size of the "
                      "built-in scratch array); split the rows over several calls", nrows, kMaxRows);
        return AA_ERR_INVALID_ARG;
    }
    if (nt < 0 || row_pitch < nt) { aa::set_error("aa_row_moments_static: need 0 <= nt <= row_pitch (nt = %lld, row_pitch = %lld)", (long long)nt, (long long)row_pitch); return AA_ERR_INVALID_ARG; }
    if (nrows == 0) return AA_OK;
    if (!device_D || !host_sum_d || !host_sum_td) { aa::set_error("aa_row_moments_static: NULL pointer argument"); return AA_ERR_INVALID_ARG; }

    u64* scratch = nullptr;
    const aa_status st = scratch_of_current_device(&scratch);
    if (st != AA_OK) return st;
    cudaStream_t cs = (cudaStream_t)stream;
    const size_t bytes = (size_t)nrows * sizeof(u64);

    /* the sums are accumulated with atomics, and the array still holds the previous call's: clear the words of this call */
    cudaError_t e;
    k_clear_moment_scratch<<<(unsigned)((nrows + kThreads - 1) / kThreads), kThreads, 0, cs>>>(nrows);
    if ((e = cudaGetLastError()) != cudaSuccess) return aa::cuda_fail(e, "aa_row_moments_static: clearing the scratch");
    if (nt > 0) {
        long long nslices = (nt + kSliceMin - 1) / kSliceMin;
        if (nslices > kMaxSlices) nslices = kMaxSlices;
        const long long slice_len = (nt + nslices - 1) / nslices;
        const dim3 grid((unsigned)((nt + slice_len - 1) / slice_len), (unsigned)nrows);
        k_row_moments_sliced<<<grid, kThreads, 0, cs>>>(device_D, (long long)row_pitch, (long long)nt, slice_len, scratch);
        if ((e = cudaGetLastError()) != cudaSuccess) return aa::cuda_fail(e, "aa_row_moments_static: kernel launch");
    }
    if ((e = cudaMemcpyAsync(host_sum_d, scratch, bytes, cudaMemcpyDeviceToHost, cs)) != cudaSuccess) return aa::cuda_fail(e, "aa_row_moments_static: D2H");
    if ((e = cudaMemcpyAsync(host_sum_td, scratch + kMaxRows, bytes, cudaMemcpyDeviceToHost, cs)) != cudaSuccess) return aa::cuda_fail(e, "aa_row_moments_static: D2H");
    if ((e = cudaStreamSynchronize(cs)) != cudaSuccess) return aa::cuda_fail(e, "aa_row_moments_static: cudaStreamSynchronize");
    return AA_OK;
}
