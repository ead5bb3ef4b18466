/*
 * k_common.cuh — device helpers shared by the K1 kernels (k_misc.cu, k_input16.cu): the exception records of the offset forms
 * (x_b = lo + off_c + r, k_misc.cu "Offset-uint8 form").
 */
#ifndef AA_K_COMMON_CUH
#define AA_K_COMMON_CUH

#include <cuda_runtime.h>
#include <stdint.h>

namespace {

/* Exception record (64 bits): channel (16 bits), residual r (20 bits, two's complement: |r| <= 65535 * 8), binned sample t (28
 * bits; aa_strategy_setup keeps chunk rows below 2^28 samples). */
__device__ __forceinline__ uint2 make_exception(int chan, long long t, int r) {
    return make_uint2((uint32_t)chan | (((uint32_t)r & 0xFFFFu) << 16), (uint32_t)t | ((((uint32_t)r >> 16) & 0xFu) << 28));
}

/* Append one exception record. The lanes of a warp that arrive together share ONE atomic on the counter; once the counter
 * has passed `cap` the chunk is bound for the other route anyway (every route test is `counter > limit`, limit <= cap, and
 * the counter never decreases), so nothing more is counted or recorded: a dense input costs one L2 read per exception
 * instead of one same-address atomic. */
__device__ __forceinline__ void append_exception(uint2* __restrict__ exc, unsigned* __restrict__ cnt, unsigned cap, uint2 rec) {
    if (*reinterpret_cast<volatile unsigned*>(cnt) > cap) return;
    const unsigned m = __activemask();
    const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    unsigned base = 0;
    if (lane == leader) base = atomicAdd(cnt, (unsigned)__popc(m));
    base = __shfl_sync(m, base, leader);
    const unsigned idx = base + (unsigned)__popc(m & ((1u << lane) - 1u));
    if (idx < cap) exc[idx] = rec;
}

}  // namespace

#endif
