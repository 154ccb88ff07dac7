// image_kernels.cuh - the pointwise steps of an MLEM iteration (sm_100a): sensitivity image, pre-pass, finalise.
//
//   sensitivity_kernel    s(y,z) of Eq. 4, evaluated in fp64, rounded once to fp32, clamped >= 0
//   prepass_kernel        wT = s * rho_in, stored TRANSPOSED (y fastest) - the s(i) rho(i) factor of Eq. 3's
//                         denominator; zeroes the transposed accumulator and the counters
//   finalise_kernel       rho_out = rho_in * acc where s > 0 else 0 (Eq. 3); acc is the sum of up to kMaxPeers
//                         accumulators - the shards of an event list split over GPUs ("each thread writes
//                         to its own copy of rho_new ... added at the end of the iteration", lifted to devices), read
//                         over NVLink peer mappings; one accumulator for the single-GPU path
#pragma once
#include "common.cuh"

namespace jpet {

constexpr int kMaxPeers = 16;
struct PeerAcc { const float* acc[kMaxPeers]; int n; };

__global__ void sensitivity_kernel(float* __restrict__ s, int n_y, int n_z, double px, double R, double L) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_y * n_z) return;
    int iy = i / n_z, iz = i - iy * n_z;
    double y = ((double)iy - 0.5 * (double)(n_y - 1)) * px;
    double z = ((double)iz - 0.5 * (double)(n_z - 1)) * px;
    double hi = fmin((0.5 * L - z) / (R - y), (0.5 * L + z) / (R + y));
    double lo = fmax(-(0.5 * L + z) / (R - y), (-0.5 * L + z) / (R + y));
    double v = (atan(hi) - atan(lo)) * 0.318309886183790671537767526745;   // Eq. 4
    s[i] = v > 0.0 ? (float)v : 0.f;
}

// wT[iz * n_y + iy] = s[iy * n_z + iz] * rho_in[...]; accT = 0; counters = 0
__global__ void prepass_kernel(const float* __restrict__ s, const float* __restrict__ rho_in, float* __restrict__ wT,
                               float* __restrict__ accT, int n_y, int n_z, unsigned long long* __restrict__ counters) {
    pdl_wait();
    int i = blockIdx.x * blockDim.x + threadIdx.x;   // transposed index: consecutive threads = consecutive iy
    if (i < n_y * n_z) {
        int iz = i / n_y, iy = i - iz * n_y;
        int src = iy * n_z + iz;
        wT[i] = s[src] * rho_in[src];
        accT[i] = 0.f;
    }
    if (i < 4) counters[i] = 0ull;
}

__global__ void finalise_kernel(const float* __restrict__ s, const float* rho_in, const __grid_constant__ PeerAcc peers,
                                float* rho_out, int n_y, int n_z) {
    pdl_wait();
    int i = blockIdx.x * blockDim.x + threadIdx.x;   // row-major index
    if (i >= n_y * n_z) return;
    int iy = i / n_z, iz = i - iy * n_z;
    const int t = iz * n_y + iy;
    float acc = 0.f;
    for (int q = 0; q < peers.n; ++q) acc += peers.acc[q][t];      // fixed order: every rank gets the same bits
    rho_out[i] = s[i] > 0.f ? rho_in[i] * acc : 0.f;
}

__global__ void ones_kernel(float* x, int M) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) x[i] = 1.f;
}

}  // namespace jpet
