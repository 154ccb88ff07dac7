// mlem_direct.cuh - the direct event kernel (sm_100a) and the evaluation counter.
//
// mlem_rows_direct_kernel handles the events of the "direct" bin (rare: non-finite, extreme angles, far outside the
// image, a row count the task table does not hold), or every event when a region does not fit shared memory: one warp
// per event, thread <-> row, w read from the global transposed image, back-projection with red.global.add.f32,
// P recomputed in the second pass.  Simple on purpose: it is the correctness path.
//
// EXACT = true is the exact-kernel mode: Eq. 7 is the saddle-point approximation of
//     P(e~ | y, z) = int_{-pi/2}^{pi/2} dtheta / pi  N(e~; e(y, z, theta), C)                     (R15)
// with e(y, z, theta) = (z + (R - y) tan, z - (R + y) tan, -2 y / cos) the exact measurement of an emission at (y, z)
// along theta; the mode evaluates the integral itself on the same 3-sigma pixel set.  In tau = tan
// theta (dtheta = dtau / (1 + tau^2)) the integrand is a near-Gaussian centred at tau* = t - sec2 b.C^-1.a / D with
// standard deviation sec2 / sqrt(D) (the ingredients of Eq. 7), so the trapezoid rule with n_nodes nodes over
// tau* +- 8 sigma converges exponentially.  With d = e(theta) - e~ = b + e(theta) - e(theta~) (b of Eq. 10):
//     d1 = u + (R - y) dtau,  d2 = u - (R + y) dtau,  d3 = -2 dy sec - 2 y (sec(theta) - sec),   dtau = tau - t,
// sec(theta) - sec = dtau (tau + t) / (sec(theta) + sec) without cancellation.  The constant prefactor of the normal
// density cancels in Eq. 3 and is dropped like K of Eq. 7.
#pragma once
#include "common.cuh"

namespace jpet {

__device__ __forceinline__ float exact_value(const RowConsts& rc, const EventConsts& e, float y, float dy, float jf, const DevParams& p,
                                             int n_nodes) {
    const float u = fmaf(jf, p.px, rc.u0);
    const float ba = fmaf(rc.alphas, u, rc.betas) * (1.f / kSqrtLH), D = fmaf(rc.eps, u, rc.delta);
    const float sec = sqrtf(e.sec2);
    const float sig = e.sec2 * rsqrtf(D), tau_c = e.t - e.sec2 * ba / D;
    const float h = 16.f * sig / (float)(n_nodes - 1);
    const float iu = 0.5f * (e.S - e.Dl), id = 0.5f * (e.S + e.Dl), il2 = 0.25f * p.c2k, g2 = 0.5f * p.gB / p.R;     // 2 gamma
    const float b3 = -2.f * dy * sec, ym = p.R - y, yp = p.R + y;
    float sum = 0.f;
    for (int k = 0; k < n_nodes; ++k) {
        const float tau = fmaf((float)k - 0.5f * (float)(n_nodes - 1), h, tau_c);
        const float dt = tau - e.t, s2 = fmaf(tau, tau, 1.f), sk = sqrtf(s2);
        const float ds = dt * (tau + e.t) / (sk + sec);
        const float d1 = fmaf(ym, dt, u), d2 = fmaf(-yp, dt, u), d3 = fmaf(-2.f * y, ds, b3);
        const float chi2 = fmaf(iu * d1, d1, fmaf(id * d2, d2, fmaf(il2 * d3, d3, g2 * (d1 - d2) * d3)));
        sum += ex2_approx(-kLH * chi2) / s2;
    }
    return h * sum;
}

template <bool EXACT>
__device__ __forceinline__ float pixel_value(const RowConsts& rc, const EventConsts& e, int iy, int j, const DevParams& p, int n_nodes) {
    if constexpr (EXACT) {
        const float y = fmaf((float)iy, p.px, p.y0);
        return exact_value(rc, e, y, y - e.y_t, (float)j, p, n_nodes);
    } else {
        return kernel_value(rc, (float)j, p.px);
    }
}

template <bool EXACT>
__global__ void __launch_bounds__(128)
mlem_rows_direct_kernel(const float* __restrict__ sorted, int stride, int* __restrict__ meta,
                        const __grid_constant__ DevParams p, const float* __restrict__ wT, float* __restrict__ accT,
                        unsigned long long* __restrict__ counters, int n_nodes) {
    pdl_wait();
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
    const int start = meta[kMetaDirectStart], count = meta[kMetaDirectCount];
    unsigned long long my_evals = 0, my_skipped = 0;
    for (int q = warp; q < count; q += n_warps) {
        const float* ev = sorted + (size_t)stride * (size_t)(start + q);      // raw triple at the head of the slot
        const EventConsts e = event_setup(__ldg(ev), __ldg(ev + 1), __ldg(ev + 2), p);
        int iy_lo, nrows;
        event_rows(e, 0, p.n_y - 1, iy_lo, nrows);
        float denom = 0.f;
        for (int r = lane; r < nrows; r += 32) {
            const RowConsts rc = row_setup(e, iy_lo + r, 0, p.n_z - 1, p);
            const float* wp = wT + (size_t)rc.lo * p.n_y + (iy_lo + r);
            my_evals += (unsigned long long)rc.len;
            for (int j = 0; j < rc.len; ++j) denom = fmaf(pixel_value<EXACT>(rc, e, iy_lo + r, j, p, n_nodes), __ldg(wp + (size_t)j * p.n_y), denom);
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) denom += __shfl_xor_sync(0xffffffffu, denom, d);
        const bool ok = (denom > 0.f) && (denom < 3.0e38f);
        if (lane == 0 && !ok) my_skipped += 1ull;
        if (!ok) continue;
        const float inv = 1.f / denom;
        for (int r = lane; r < nrows; r += 32) {
            const RowConsts rc = row_setup(e, iy_lo + r, 0, p.n_z - 1, p);
            float* ap = accT + (size_t)rc.lo * p.n_y + (iy_lo + r);
            for (int j = 0; j < rc.len; ++j) red_add_f32(ap + (size_t)j * p.n_y, pixel_value<EXACT>(rc, e, iy_lo + r, j, p, n_nodes) * inv);
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) my_evals += __shfl_xor_sync(0xffffffffu, my_evals, d);
    if (lane == 0 && my_evals) atomicAdd(counters + 0, my_evals);
    if (lane == 0 && my_skipped) atomicAdd(counters + 1, my_skipped);
    // this kernel always follows the tiled event kernel(s) in the stream: reset the work counters for the next run over
    // the same sorted events (jpet_reconstruct sorts once and iterates)
    if (blockIdx.x == 0 && threadIdx.x == 0) { meta[kMetaCounter0] = 0; meta[kMetaCounter1] = 0; }
}

// |E_j| only (jpet_count_evals): thread per event, rows in a loop, no kernel values.
__global__ void count_evals_kernel(const float* __restrict__ events, long long n, const __grid_constant__ DevParams p,
                                   unsigned long long* __restrict__ counters) {
    unsigned long long evals = 0, skipped = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        EventConsts e = event_setup(events[3 * i], events[3 * i + 1], events[3 * i + 2], p);
        int iy_lo, nrows, cnt = 0;
        event_rows(e, 0, p.n_y - 1, iy_lo, nrows);
        for (int r = 0; r < nrows; ++r) cnt += row_setup(e, iy_lo + r, 0, p.n_z - 1, p).len;
        evals += cnt;
        skipped += cnt == 0;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        evals += __shfl_xor_sync(0xffffffffu, evals, d);
        skipped += __shfl_xor_sync(0xffffffffu, skipped, d);
    }
    if ((threadIdx.x & 31) == 0) {
        if (evals) atomicAdd(counters + 0, evals);
        if (skipped) atomicAdd(counters + 1, skipped);
    }
}

}  // namespace jpet
