// kf_wside.cuh -- W-node stages (QKV projection, W_O, FFN) and the M-microbatch inter-layer pipeline: shared
// declarations of kf_wgemm.cu (the tcgen05 weight-streaming GEMM) and kf_wside.cu (the C ABI).  Product code.
#pragma once

#include <cuda.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/kflume.h"

namespace kf {

constexpr int kWgBK = 64;        // halfs per k-block = one 128-byte swizzle row
constexpr int kWgTileN = 128;    // output features per CTA = UMMA M = TMEM lanes
constexpr int kWgThreads = 192;  // warp 0: TMA producer; warp 1: TMEM allocator + MMA issuer; warps 2..5: epilogue
constexpr int kWgMaxBatch = 128;
constexpr int kWgMaxCtas = 160;   // upper bound of the persistent grid (SM count)

__host__ __device__ constexpr int wgemm_stages(int nb, bool dual) { return dual ? (nb > 64 ? 4 : 5) : (nb > 64 ? 6 : 8); }
__host__ __device__ constexpr int wgemm_smem_bytes(int nb, bool dual) {
    return wgemm_stages(nb, dual) * (kWgTileN * kWgBK * 2 * (dual ? 2 : 1) + nb * kWgBK * 2) + 1024;
}

struct WGemmArgs {
    int K, N, B;          // reduction length, output features (per accumulator), valid batch rows
    int nkb;              // k-blocks (of 64) per tile = K / 64
    int n_ctas;           // persistent grid: CTA c owns k-blocks [c * per, (c + 1) * per) of the (tile, k-block) sequence
    int seg_end[3];       // output segments: features [seg_end[i-1], seg_end[i]) go to out[i] (boundaries % 128 == 0)
    int ld[3];            // row stride (halfs) of each output
    __half *out[3];
    float *partial;       // [n_ctas][2 slots][1 or 2][NB][128] fp32: pieces of tiles shared between spans
    int up_row_offset;    // dual kernel: row of the first `up` weight in the weight tensor (gate rows come first)
};

// returns the number of kernels launched (1) or a negative KF_E* code
// pdl: launch programmatically dependent on the preceding kernel of the stream (the kernel sets up barriers, TMEM and
// descriptors, then waits for that kernel to complete before it touches global memory)
int launch_wgemm(const CUtensorMap &tmW, const CUtensorMap &tmX, const WGemmArgs &a, int nb, bool dual, bool pdl,
                 cudaStream_t s);
int launch_cast_o(const float *o, __half *o16, size_t n, cudaStream_t s);

}  // namespace kf
