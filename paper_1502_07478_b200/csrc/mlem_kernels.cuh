// mlem_kernels.cuh - sm_100a device code of the list-mode MLEM hot path (arXiv:1502.07478).
//
// Citations are /root/reference/PAPER.md lines.  Nothing here is shared with oracle/.
//
// Kernels
//   sensitivity_kernel    s(y,z) of Eq. 4, evaluated in fp64, rounded once to fp32, clamped >= 0
//   prepass_kernel        w = s * rho_in (the s(i) rho(i) factor of Eq. 3's denominator);
//                         zeroes the accumulator replicas
//   mlem_events_kernel    steps 1-3: Eq. 2, 3-sigma ellipse rows (App. B
//                         :251-267), kernel of Eq. 7-12, denominator, scatter
//   finalise_kernel       acc = sum of replicas; rho_out = rho_in * acc where s > 0 else 0 (Eq. 3)
//
// Algebra used by mlem_events_kernel (diagonal C^-1 = diag(iz2, iz2, il2), iz2 = 1/sigma_z^2,
// il2 = 1/sigma_dl^2; t = tan theta~, sec2 = 1 + t^2; pixel centre (y, z); dy = y - y~, dz = z - z~;
// u = dz - t dy; k = a3 coefficient).  With o, a, b of Eq. 8-10 written out, the four quadratic forms are
//   b.C^-1.b = 2 iz2 u^2 + 4 il2 sec2 dy^2                                              (B.3)
//   b.C^-1.a = -2 iz2 sec2 y u + 2 k il2 sec2 t y dy
//   a.C^-1.a = 2 iz2 sec2^2 (y^2 + R^2) + k^2 il2 sec2 t^2 y^2
//   o.C^-1.b = -2 iz2 sec2 t y u + 2 il2 sec2 (1 + 2 t^2) y dy
// so along one image row (fixed y) everything is a polynomial in u:
//   q  = b.C^-1.b = c1 u^2 + c2          ba = b.C^-1.a = alpha u + beta
//   D  = a.C^-1.a + 2 o.C^-1.b = eps u + delta
//   P  = K D^-1/2 exp(-1/2 (q - ba^2 / D))                                                (Eq. 7)
// K (the constant prefactor) cancels between numerator and denominator of Eq. 3 and is dropped.
// The exponent is evaluated in base 2: constants carry the factor LH = log2(e)/2 (alpha, beta carry
// sqrt(LH)), so P = r * ex2(c1s u^2 + c2s + (ba_s r)^2) with r = rsqrt(D): 8 FP32 + 2 MUFU per pixel.
// Row r of the ellipse is the closed interval |u| <= sqrt((9 - c2)/c1) (B.3 solved for dz), so pixels are
// enumerated by row spans and no lane is spent on a failed ellipse test (the paper's bbox + test wastes
// about one third of the lanes).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace jpet {

struct DevParams {
    // grid
    int n_y, n_z;
    float px, inv_px, y0, z0;          // y0/z0: centre of pixel row/column 0
    // geometry and kernel constants
    float inv2R, R2;
    float hy_coef;                     // 1.5 sigma_dl: half-height of the ellipse is hy_coef * cos(theta~)
    float half_sz2;                    // sigma_z^2 / 2 = 1 / c1
    float c1s;                         // -LH * 2 iz2
    float c2k;                         // 4 il2          (c2 = c2k * sec2 * dy^2)
    float ak;                          // -2 iz2         (alpha = ak sec2 y)
    float bk;                          // 2 k il2        (beta = bk sec2 t y dy)
    float d1k;                         // 2 iz2          (delta term sec2^2 (y^2 + R^2))
    float d2k;                         // k^2 il2        (delta term sec2 t^2 y^2)
    float d3k;                         // 4 il2          (delta term sec2 (1 + 2 t^2) y dy)
    // table capacities (per event group)
    int nrow_max, nseg_max;
};

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ void red_add_f32(float* addr, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void group_barrier(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

constexpr float kLH = 0.72134752044448170368f;       // log2(e) / 2
constexpr float kSqrtLH = 0.84932180028801904272f;   // sqrt(log2(e) / 2)

// ------------------------------------------------------------------------------------------------------
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

__global__ void prepass_kernel(const float* __restrict__ s, const float* __restrict__ rho_in, float* __restrict__ w,
                               float* __restrict__ acc, int M, int n_rep, unsigned long long* __restrict__ counters) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) {
        w[i] = s[i] * rho_in[i];
        for (int r = 0; r < n_rep; ++r) acc[(size_t)r * M + i] = 0.f;
    }
    if (i < 2) counters[i] = 0ull;
}

__global__ void finalise_kernel(const float* __restrict__ s, const float* rho_in, const float* __restrict__ acc,
                                float* rho_out, int M, int n_rep) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= M) return;
    float a = 0.f;
    for (int r = 0; r < n_rep; ++r) a += acc[(size_t)r * M + i];
    rho_out[i] = s[i] > 0.f ? rho_in[i] * a : 0.f;
}

__global__ void ones_kernel(float* x, int M) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) x[i] = 1.f;
}

// ------------------------------------------------------------------------------------------------------
// Per-row record of the current event (shared memory, one table per event group).
struct __align__(16) RowRec {
    float u0;      // u at the first pixel of the row
    float c2s;     // -LH * c2
    float betas;   // sqrt(LH) * beta
    float delta;
    float alphas;  // sqrt(LH) * alpha
    float eps;
    int base;      // linear pixel index of the first pixel of the row
    int len;       // pixels in the row
};

struct EventConsts {
    float t, sec2, y_t, z_t;
    int iy_lo, nrows;   // nrows == 0: event skipped
};

// Eq. 2 and the row range of the 3-sigma ellipse.
__device__ __forceinline__ EventConsts event_setup(float zu, float zd, float dl, const DevParams& p) {
    EventConsts e;
    e.t = (zu - zd) * p.inv2R;                      // tan theta~
    e.sec2 = fmaf(e.t, e.t, 1.f);
    float cos_t = rsqrtf(e.sec2);
    e.y_t = -0.5f * dl * cos_t;                     // y~
    e.z_t = fmaf(e.y_t, e.t, 0.5f * (zu + zd));     // z~
    float hy = p.hy_coef * cos_t;                   // 3 sigma_y, sigma_y = sigma_dl cos(theta~) / 2
    float flo = (e.y_t - hy - p.y0) * p.inv_px;
    float fhi = (e.y_t + hy - p.y0) * p.inv_px;
    bool finite = (fabsf(zu) < 1e30f) && (fabsf(zd) < 1e30f) && (fabsf(dl) < 1e30f);   // false for NaN too
    flo = fminf(fmaxf(flo, -1.f), (float)p.n_y);
    fhi = fminf(fmaxf(fhi, -1.f), (float)p.n_y);
    int lo = max(0, __float2int_ru(flo));
    int hi = min(p.n_y - 1, __float2int_rd(fhi));
    e.iy_lo = lo;
    e.nrows = finite ? max(0, hi - lo + 1) : 0;
    e.nrows = min(e.nrows, p.nrow_max);
    return e;
}

__device__ __forceinline__ RowRec row_setup(const EventConsts& e, int iy, const DevParams& p) {
    RowRec r;
    float y = fmaf((float)iy, p.px, p.y0);
    float dy = y - e.y_t;
    float c2 = p.c2k * e.sec2 * dy * dy;
    float rem = 9.f - c2;                                  // row chord: c1 u^2 <= 9 - c2
    float hw = sqrtf(fmaxf(rem, 0.f) * p.half_sz2);
    float zc = fmaf(e.t, dy, e.z_t);                       // u = 0 on the line z = z~ + t dy
    float flo = fminf(fmaxf((zc - hw - p.z0) * p.inv_px, -1.f), (float)p.n_z);
    float fhi = fminf(fmaxf((zc + hw - p.z0) * p.inv_px, -1.f), (float)p.n_z);
    int lo = max(0, __float2int_ru(flo));
    int hi = min(p.n_z - 1, __float2int_rd(fhi));
    int len = rem >= 0.f ? max(0, hi - lo + 1) : 0;
    float ysec = y * e.sec2;
    float alpha = p.ak * ysec;
    r.u0 = fmaf((float)lo, p.px, p.z0) - zc;
    r.c2s = -kLH * c2;
    r.betas = kSqrtLH * p.bk * ysec * e.t * dy;
    r.delta = p.d1k * e.sec2 * e.sec2 * fmaf(y, y, p.R2) + p.d2k * ysec * e.t * e.t * y
              + p.d3k * ysec * fmaf(2.f * e.t, e.t, 1.f) * dy;
    r.alphas = kSqrtLH * alpha;
    r.eps = 2.f * e.t * alpha;
    r.base = iy * p.n_z + lo;
    r.len = len;
    return r;
}

// P (up to the constant K) at offset j of a row.
__device__ __forceinline__ float kernel_value(const RowRec& r, float jpx, float c1s) {
    float u = r.u0 + jpx;
    float e2 = fmaf(c1s * u, u, r.c2s);
    float ba = fmaf(r.alphas, u, r.betas);
    float D = fmaf(r.eps, u, r.delta);
    float rs = rsqrt_approx(D);
    float bar = ba * rs;
    e2 = fmaf(bar, bar, e2);
    return rs * ex2_approx(e2);
}

// One event group = NW warps working on one event at a time.  A "segment" is W consecutive pixels of one
// ellipse row; a warp evaluates 32/W segments per iteration.  The first NIT iterations keep P in
// registers for the scatter pass; later iterations (events larger than the tuned capacity) recompute it.
template <int W, int NW, int NIT, int THREADS>
__global__ void __launch_bounds__(THREADS)
mlem_events_kernel(const float* __restrict__ events, long long n, const __grid_constant__ DevParams p,
                   const float* __restrict__ w, float* __restrict__ acc, long long rep_stride, int n_rep,
                   unsigned long long* __restrict__ counters) {
    constexpr int G = 32 / W;
    constexpr int GT = NW * 32;
    constexpr int GROUPS = THREADS / GT;
    constexpr int SEG_PER_IT = G * NW;
    static_assert(THREADS % GT == 0 && 32 % W == 0, "bad shape");

    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int group = threadIdx.x / GT;
    const int gtid = threadIdx.x % GT;
    const int lane = threadIdx.x & 31;
    const int warp_in_group = gtid >> 5;
    // per-group layout: RowRec[nrow_max] | uint32 segmap[nseg_max] | float red[NW]
    const size_t rows_bytes = (size_t)p.nrow_max * sizeof(RowRec);
    const size_t seg_bytes = (((size_t)p.nseg_max * 4 + 15) / 16) * 16;
    const size_t group_bytes = rows_bytes + seg_bytes + 16 * ((NW * 4 + 15) / 16);
    unsigned char* gbase = smem_raw + group * group_bytes;
    RowRec* rowtab = reinterpret_cast<RowRec*>(gbase);
    uint32_t* segmap = reinterpret_cast<uint32_t*>(gbase + rows_bytes);
    float* red = reinterpret_cast<float*>(gbase + rows_bytes + seg_bytes);

    float* acc_rep = acc + (size_t)(blockIdx.x % n_rep) * rep_stride;
    const int sub = lane / W;                       // sub-warp (segment slot) within the warp
    const int jl = lane % W;                        // pixel within the segment
    const float jlpx = (float)jl * p.px;
    const float wpx = (float)W * p.px;

    unsigned long long my_evals = 0, my_skipped = 0;
    const long long n_groups = (long long)gridDim.x * GROUPS;

    for (long long ev = (long long)blockIdx.x * GROUPS + group; ev < n; ev += n_groups) {
        // ---- step 1: Eq. 2 + row range (all lanes, broadcast loads) -----------------------------------
        const float zu = __ldg(events + 3 * ev), zd = __ldg(events + 3 * ev + 1), dl = __ldg(events + 3 * ev + 2);
        const EventConsts e = event_setup(zu, zd, dl, p);

        // ---- row table + segment map (threads <-> rows) ------------------------------------------------
        int seg_total = 0, px_total = 0;
        for (int r0 = 0; r0 < e.nrows; r0 += GT) {
            int r = r0 + gtid;
            int nseg = 0, len = 0;
            RowRec rec;
            if (r < e.nrows) {
                rec = row_setup(e, e.iy_lo + r, p);
                len = rec.len;
                nseg = (len + W - 1) / W;
                rowtab[r] = rec;
            }
            // exclusive scan of nseg over the group's threads
            int incl = nseg, lsum = len;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                int v = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += v;
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) lsum += __shfl_xor_sync(0xffffffffu, lsum, d);
            int warp_off = 0, chunk_total = __shfl_sync(0xffffffffu, incl, 31), chunk_px = lsum;
            if (NW > 1) {   // combine the warps of the group
                __shared__ int scan_buf[THREADS / 32][2];
                if (lane == 31) { scan_buf[threadIdx.x >> 5][0] = incl; scan_buf[threadIdx.x >> 5][1] = lsum; }
                group_barrier(1 + group, GT);
                chunk_total = 0; chunk_px = 0;
#pragma unroll
                for (int k = 0; k < NW; ++k) {
                    int v = scan_buf[group * NW + k][0];
                    if (k < warp_in_group) warp_off += v;
                    chunk_total += v;
                    chunk_px += scan_buf[group * NW + k][1];
                }
                group_barrier(1 + group, GT);
            }
            int excl = seg_total + warp_off + incl - nseg;
            for (int s = 0; s < nseg; ++s)
                if (excl + s < p.nseg_max) segmap[excl + s] = (uint32_t)r | ((uint32_t)s << 16);
            seg_total += chunk_total;
            px_total += chunk_px;
        }
        seg_total = min(seg_total, p.nseg_max);
        if (NW > 1) group_barrier(1 + group, GT); else __syncwarp();

        // ---- step 2: kernel values + denominator --------------------------------------------------------
        float preg[NIT];
        int ireg[NIT];
        float denom = 0.f;
        const int my_first = warp_in_group * G + sub;
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            int sidx = it * SEG_PER_IT + my_first;
            float P = 0.f;
            int idx = -1;
            if (sidx < seg_total) {
                uint32_t m = segmap[sidx];
                const RowRec rec = rowtab[m & 0xffffu];
                int j = (int)(m >> 16) * W + jl;
                if (j < rec.len) {
                    P = kernel_value(rec, fmaf((float)(m >> 16), wpx, jlpx), p.c1s);
                    idx = rec.base + j;
                    denom = fmaf(P, __ldg(w + idx), denom);
                }
            }
            preg[it] = P;
            ireg[it] = idx;
        }
        for (int sidx = NIT * SEG_PER_IT + my_first; sidx < seg_total; sidx += SEG_PER_IT) {   // overflow, uncached
            uint32_t m = segmap[sidx];
            const RowRec rec = rowtab[m & 0xffffu];
            int j = (int)(m >> 16) * W + jl;
            if (j < rec.len) {
                float P = kernel_value(rec, fmaf((float)(m >> 16), wpx, jlpx), p.c1s);
                denom = fmaf(P, __ldg(w + rec.base + j), denom);
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) denom += __shfl_xor_sync(0xffffffffu, denom, d);
        if (NW > 1) {
            if (lane == 0) red[warp_in_group] = denom;
            group_barrier(1 + group, GT);
            denom = 0.f;
#pragma unroll
            for (int k = 0; k < NW; ++k) denom += red[k];
        }

        // ---- step 3: scatter P / denominator -------------------------------------------------------------
        const bool ok = (seg_total > 0) && (denom > 0.f) && (denom < 3.0e38f);
        if (ok) {
            const float inv = 1.f / denom;
#pragma unroll
            for (int it = 0; it < NIT; ++it)
                if (ireg[it] >= 0) red_add_f32(acc_rep + ireg[it], preg[it] * inv);
            for (int sidx = NIT * SEG_PER_IT + my_first; sidx < seg_total; sidx += SEG_PER_IT) {
                uint32_t m = segmap[sidx];
                const RowRec rec = rowtab[m & 0xffffu];
                int j = (int)(m >> 16) * W + jl;
                if (j < rec.len) {
                    float P = kernel_value(rec, fmaf((float)(m >> 16), wpx, jlpx), p.c1s);
                    red_add_f32(acc_rep + rec.base + j, P * inv);
                }
            }
        }
        if (gtid == 0) {
            my_evals += (unsigned long long)px_total;
            my_skipped += ok ? 0ull : 1ull;
        }
        // tables are rewritten by the next event: everyone must be done reading them
        if (NW > 1) group_barrier(1 + group, GT); else __syncwarp();
    }
    if (gtid == 0) {
        if (my_evals) atomicAdd(counters + 0, my_evals);
        if (my_skipped) atomicAdd(counters + 1, my_skipped);
    }
}

// |E_j| only (jpet_count_evals): thread per event, rows in a loop, no kernel values.
__global__ void count_evals_kernel(const float* __restrict__ events, long long n, const __grid_constant__ DevParams p,
                                   unsigned long long* __restrict__ counters) {
    unsigned long long evals = 0, skipped = 0;
    for (long long ev = (long long)blockIdx.x * blockDim.x + threadIdx.x; ev < n; ev += (long long)gridDim.x * blockDim.x) {
        EventConsts e = event_setup(events[3 * ev], events[3 * ev + 1], events[3 * ev + 2], p);
        int cnt = 0;
        for (int r = 0; r < e.nrows; ++r) cnt += row_setup(e, e.iy_lo + r, p).len;
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
