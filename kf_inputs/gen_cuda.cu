// gen_cuda.cu -- device twin of kf_inputs/gen.py.  Fills fp16 tensors with the SAME
// stateless values as the numpy generator, bit for bit, so that GPU-resident workloads too large to stage
// through the host (cfg 3-5) see exactly the inputs the oracle sees.  Holds none of the method's arithmetic;
// it is a separate library (libkfgen.so) and links nothing from libkflume.
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__host__ __device__ inline uint64_t mix64(uint64_t z) {
    z ^= z >> 30;
    z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27;
    z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}
__host__ __device__ inline uint64_t stream_key(uint64_t seed, uint64_t stream) {
    return mix64(seed ^ (stream * 0xD1B54A32D192ED03ull));
}
__device__ inline __half normal16(uint64_t x) {
    // sum of the 8 bytes, via two SAD-like steps
    uint32_t lo = (uint32_t)x, hi = (uint32_t)(x >> 32);
    int s = (int)(__vsadu4(lo, 0u) + __vsadu4(hi, 0u));
    const float c = __uint_as_float(0x3B9CC4BFu);
    return __float2half_rn(__fmul_rn((float)(s - 1020), c));
}
__device__ inline uint64_t make_idx(uint64_t layer, uint64_t req, uint64_t pos, uint64_t head, uint64_t dim) {
    return dim | (head << 7) | (pos << 14) | (req << 38) | (layer << 54);
}

// out[heads][n_pos][128]; one thread = 8 consecutive dims (one 16-byte store)
__global__ void fill_kernel(uint64_t key, int layer, int req, int64_t pos_begin, int64_t n_pos, int heads,
                            __half *out) {
    const int64_t total = (int64_t)heads * n_pos * 16;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (int64_t)gridDim.x * blockDim.x) {
        const int c = (int)(i & 15);
        const int64_t row = i >> 4;
        const int64_t t = row % n_pos;
        const int h = (int)(row / n_pos);
        __align__(16) __half v[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const uint64_t idx = make_idx(layer, req, pos_begin + t, h, c * 8 + e);
            v[e] = normal16(mix64(key + (idx + 1) * 0x9E3779B97F4A7C15ull));
        }
        *reinterpret_cast<int4 *>(out + row * 128 + c * 8) = *reinterpret_cast<const int4 *>(v);
    }
}

// out[B][heads][128]; row r uses position pos[r] (pos[r] < 0: row left untouched)
__global__ void fill_rows_kernel(uint64_t key, int layer, const int32_t *pos, int B, int heads, __half *out) {
    const int total = B * heads * 16;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        const int c = i & 15, row = i >> 4;
        const int h = row % heads, r = row / heads;
        const int ps = pos[r];
        if (ps < 0) continue;
        __align__(16) __half v[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            const uint64_t idx = make_idx(layer, r, ps, h, c * 8 + e);
            v[e] = normal16(mix64(key + (idx + 1) * 0x9E3779B97F4A7C15ull));
        }
        *reinterpret_cast<int4 *>(out + (size_t)row * 128 + c * 8) = *reinterpret_cast<const int4 *>(v);
    }
}

}  // namespace

extern "C" {

// Fill out[heads][n_pos][128] (device, fp16) with stream `stream_id` values of (layer, req) at positions
// pos_begin .. pos_begin + n_pos - 1.  Returns 0 or the cudaError_t of the launch.
int kfgen_fill(uint64_t seed, int stream_id, int layer, int req, int64_t pos_begin, int64_t n_pos, int heads,
               void *out, void *cuda_stream) {
    if (n_pos <= 0 || heads <= 0) return 0;
    const int64_t total = (int64_t)heads * n_pos * 16;
    int blocks = (int)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
    fill_kernel<<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>(stream_key(seed, (uint64_t)stream_id), layer, req,
                                                                pos_begin, n_pos, heads, (__half *)out);
    return (int)cudaPeekAtLastError();
}

// Fill out[B][heads][128] where row r is request r at position pos[r] (device int32 array).
int kfgen_fill_rows(uint64_t seed, int stream_id, int layer, const int32_t *pos, int B, int heads, void *out,
                    void *cuda_stream) {
    if (B <= 0 || heads <= 0) return 0;
    const int total = B * heads * 16;
    fill_rows_kernel<<<(total + 255) / 256, 256, 0, (cudaStream_t)cuda_stream>>>(
        stream_key(seed, (uint64_t)stream_id), layer, pos, B, heads, (__half *)out);
    return (int)cudaPeekAtLastError();
}
}
