// histogram.cuh - direct reconstruction (Eq. 2; Fig. 4b): every event is reconstructed to the point
// (y~, z~) and counted in the pixel that contains it.  Bandwidth-bound companion of the MLEM path: 12 bytes read per
// event, one 32-bit atomic increment.
//
// The pixel index is an integer decided by floating point, so the arithmetic is pinned: IEEE fp32, round to nearest,
// in exactly this order (no approximate MUFU, no contraction beyond the fused multiply-adds written here), whatever the
// compiler flags.  The oracle is Eq. 2 in fp64 + floor: counts agree exactly for every event farther than the fp32
// rounding error (about 2^-21 (|c| + 1) pixels) from a pixel border, the others land in an adjacent pixel (R24):
//     t   = (z_u - z_d) * inv2R                      inv2R = fp32(1 / (2 R))
//     sec = sqrt(fma(t, t, 1))
//     y~  = (-0.5 * dl) / sec                        z~ = fma(y~, t, 0.5 * (z_u + z_d))
//     iy  = floor(fma(y~, inv_px, oy))               oy = fp32((n_y - 1) / 2 + 1/2)   (likewise iz with oz)
// Events are read with coalesced 16-byte loads into a shared-memory tile (sort_kernels.cuh); images of up to
// kHistSmemMax pixels are histogrammed in shared memory per block and flushed once.
#pragma once
#include "sort_kernels.cuh"

namespace jpet {

constexpr int kHistSmemMax = 6144;     // pixels of a per-block shared-memory histogram (24 KB beside the 24 KB event tile)

struct HistParams { int n_y, n_z; float inv2R, inv_px, oy, oz; };

__device__ __forceinline__ int direct_pixel(float zu, float zd, float dl, const HistParams& h) {
    const float t = __fmul_rn(__fsub_rn(zu, zd), h.inv2R);
    const float sec = __fsqrt_rn(__fmaf_rn(t, t, 1.f));
    const float yt = __fdiv_rn(__fmul_rn(-0.5f, dl), sec);
    const float zt = __fmaf_rn(yt, t, __fmul_rn(0.5f, __fadd_rn(zu, zd)));
    const float fy = floorf(__fmaf_rn(yt, h.inv_px, h.oy)), fz = floorf(__fmaf_rn(zt, h.inv_px, h.oz));
    // NaN compares false: non-finite events fall outside
    if (!(fy >= 0.f && fy < (float)h.n_y && fz >= 0.f && fz < (float)h.n_z)) return -1;
    return (int)fy * h.n_z + (int)fz;
}

__global__ void __launch_bounds__(kBinBlock)
direct_histogram_kernel(const float* __restrict__ events, int n, const __grid_constant__ HistParams h,
                        unsigned int* __restrict__ hist, unsigned long long* __restrict__ n_outside, int use_smem) {
    extern __shared__ __align__(16) float bin_smem[];
    float* tile = bin_smem;
    unsigned int* hs = reinterpret_cast<unsigned int*>(bin_smem + 3 * kBinTile);
    const int tid = threadIdx.x, M = h.n_y * h.n_z;
    if (use_smem)
        for (int b = tid; b < M; b += kBinBlock) hs[b] = 0u;
    int outside = 0;
    // 32-bit tile offsets: the host launches at most 2^30 events at a time (jpet_direct_histogram), so base + stride stays
    // below 2^31 (a 64-bit walk cost 70 % on B200: 1.56 ms against 0.90 ms for 10^8 events)
    for (int base = blockIdx.x * kBinTile; base < n; base += gridDim.x * kBinTile) {
        __syncthreads();                                   // previous tile consumed (and the histogram zeroed)
        load_event_tile(events, n, base, tile);
        __syncthreads();
#pragma unroll
        for (int q = 0; q < kBinPer; ++q) {
            const int k = q * kBinBlock + tid;
            if (base + k < n) {
                const int px = direct_pixel(tile[3 * k], tile[3 * k + 1], tile[3 * k + 2], h);
                if (px < 0) ++outside;
                else atomicAdd(use_smem ? hs + px : hist + px, 1u);
            }
        }
    }
    if (use_smem) {
        __syncthreads();
        for (int b = tid; b < M; b += kBinBlock) {
            const unsigned int c = hs[b];
            if (c) atomicAdd(hist + b, c);
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) outside += __shfl_xor_sync(0xffffffffu, outside, d);
    if ((tid & 31) == 0 && outside) atomicAdd(n_outside, (unsigned long long)outside);
}

}  // namespace jpet
