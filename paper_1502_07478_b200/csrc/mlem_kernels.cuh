// mlem_kernels.cuh - sm_100a device code of the list-mode MLEM hot path (arXiv:1502.07478).
//
// Citations are /root/reference/PAPER.md lines.  Nothing here is shared with oracle/.
//
// Kernels
//   sensitivity_kernel    s(y,z) of Eq. 4, evaluated in fp64, rounded once to fp32, clamped >= 0
//   prepass_kernel        wT = s * rho_in, stored TRANSPOSED (y fastest) - the s(i) rho(i) factor of Eq. 3's
//                         denominator; zeroes the transposed accumulator
//   bin_*_kernel          counting sort of the events by the image sub-tile their reconstructed point
//                         (y~, z~) of Eq. 2 falls in, and the work-item list (sub-tile, chunk of events)
//   mlem_rows_kernel      steps 1-3: Eq. 2, 3-sigma ellipse rows (App. B
//                         :251-267), kernel of Eq. 7-12, denominator, back-projection
//   finalise_kernel       rho_out = rho_in * acc where s > 0 else 0 (Eq. 3)
//
// Algebra used by mlem_rows_kernel (diagonal C^-1 = diag(iz2, iz2, il2), iz2 = 1/sigma_z^2,
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
//
// Schedule of mlem_rows_kernel (B200 design, not the paper's warp-per-event/texture scheme):
//   * one CTA (NW warps) works on one event at a time; THREAD <-> ELLIPSE ROW (optionally a 1/NH part of a
//     row), so the row constants live in registers and the inner loop walks the row's pixels with no
//     table look-ups; the P values of the walk stay in registers for the back-projection pass;
//   * events are pre-sorted by image sub-tile; a CTA takes a work item (sub-tile, chunk of events), stages
//     the w = s*rho region (sub-tile + halo) in shared memory, accumulates P/denominator into a PRIVATE
//     shared-memory region with plain (non-atomic) read-modify-writes, and flushes the region once with
//     red.global.add.f32.  Measured on B200: global red.add tops out at ~2.8e10 warp requests/s, a factor 5-10
//     below what the SFU/FP32 pipes can produce, so the scatter has to stay on chip;
//   * regions are stored transposed (y fastest, row stride HS a multiple of 32): lanes are consecutive
//     image rows, so every shared-memory access of a warp is bank-conflict free whatever the ellipse tilt.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

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
    float sq, inv_sq;                  // sqrt(-c1s) and its inverse (u is rescaled so the Gaussian term is -u'^2)
    float pxs;                         // px * sq: step of u' between neighbouring pixels of a row
    float H0p;                         // 9 (sigma_z^2 / 2) / px^2: half chord^2 in pixels^2 is H0p + H2p dy^2
    float c2k;                         // 4 il2          (c2 = c2k * sec2 * dy^2)
    float ak;                          // -2 iz2         (alpha = ak sec2 y)
    float bk;                          // 2 k il2        (beta = bk sec2 t y dy)
    float d1k;                         // 2 iz2          (delta term sec2^2 (y^2 + R^2))
    float d2k;                         // k^2 il2        (delta term sec2 t^2 y^2)
    float d3k;                         // 4 il2          (delta term sec2 (1 + 2 t^2) y dy)
    // off-diagonal coefficient gamma of C^-1 (Eq. 12; 0 = the paper's diagonal case).  With
    // a1 - a2 = 2 R sec2, o1 - o2 = 2 R sec2 t, b1 = b2, b3 = -2 dy sec, a3 = -k y sec t it adds
    //   b.C^-1.a += -4 gamma R sec^3 dy,   a.C^-1.a += -4 gamma k R sec^3 t y,   o.C^-1.b += -4 gamma R sec^3 t dy
    // and leaves b.C^-1.b (the 3-sigma ellipse) unchanged.
    float gB;                          // 4 gamma R
    float gD0;                         // 4 gamma R k
    // binning and shared-memory regions (pixel units)
    int Hy, Hz;                        // halo on each side of a sub-tile
    int Sy, Sz;                        // sub-tile size
    int HS, WZ;                        // region: HS rows (y, fastest, multiple of 32) x WZ columns (z)
    int nby, nbz;                      // bins cover pixel indices [-Hy, n_y + Hy) x [-Hz, n_z + Hz)
    float t_max;                       // events with |tan theta~| above this go to the direct (global) path
    int chunk;                         // events per work item
    int nr_min, nr_max;                // third-generation kernel: ellipse row counts covered by its task table;
                                       // nr_max > 0 makes the records carry the UNCLIPPED row range of the ellipse
};

struct WorkItem { int bin, start, count; };

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
__device__ __forceinline__ float sqrt_approx(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ void red_add_f32(float* addr, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(addr), "f"(v) : "memory");
}

// Programmatic dependent launch (jpet_api.cu launches the kernels of an iteration with the stream-serialisation
// attribute): everything before this call may overlap the tail of the previous kernel in the stream; nothing that
// the previous kernel wrote is read before it.  A no-op for a kernel launched without the attribute.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

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

__global__ void finalise_kernel(const float* __restrict__ s, const float* rho_in, const float* __restrict__ accT,
                                float* rho_out, int n_y, int n_z) {
    pdl_wait();
    int i = blockIdx.x * blockDim.x + threadIdx.x;   // row-major index
    if (i >= n_y * n_z) return;
    int iy = i / n_z, iz = i - iy * n_z;
    rho_out[i] = s[i] > 0.f ? rho_in[i] * accT[iz * n_y + iy] : 0.f;
}

__global__ void ones_kernel(float* x, int M) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < M) x[i] = 1.f;
}

// ------------------------------------------------------------------------------------------------------
struct EventConsts {
    float t, sec2, y_t, z_t;
    float fy;           // y~ in pixel units (row index, fractional)
    float hy_px;        // half height of the ellipse in pixels
    bool finite;
};

// Eq. 2.
__device__ __forceinline__ EventConsts event_setup(float zu, float zd, float dl, const DevParams& p) {
    EventConsts e;
    e.t = (zu - zd) * p.inv2R;                      // tan theta~
    e.sec2 = fmaf(e.t, e.t, 1.f);
    float cos_t = rsqrt_approx(e.sec2);
    e.y_t = -0.5f * dl * cos_t;                     // y~
    e.z_t = fmaf(e.y_t, e.t, 0.5f * (zu + zd));     // z~
    e.fy = (e.y_t - p.y0) * p.inv_px;
    e.hy_px = p.hy_coef * cos_t * p.inv_px;         // 3 sigma_y / pixel, sigma_y = sigma_dl cos(theta~) / 2
    e.finite = (fabsf(zu) < 1e30f) && (fabsf(zd) < 1e30f) && (fabsf(dl) < 1e30f);   // false for NaN too
    return e;
}

// Rows of the ellipse clipped to [row_lo, row_hi]: returns first row and count.
__device__ __forceinline__ void event_rows(const EventConsts& e, int row_lo, int row_hi, int& iy_lo, int& nrows) {
    int lo = max(row_lo, __float2int_ru(e.fy - e.hy_px));      // cvt saturates; non-finite events are dropped below
    int hi = min(row_hi, __float2int_rd(e.fy + e.hy_px));
    iy_lo = lo;
    nrows = e.finite ? max(0, hi - lo + 1) : 0;
}

struct RowConsts {
    float u0;      // u at the first pixel of this thread's part of the row
    float c2s;     // -LH * c2
    float betas;   // sqrt(LH) * beta
    float delta;
    float alphas;  // sqrt(LH) * alpha
    float eps;
    int lo;        // first column of the part
    int len;       // pixels in the part
};

// Row constants and the span of row iy, clipped to columns [col_lo, col_hi]; part h of NH equal parts.
template <int NH>
__device__ __forceinline__ RowConsts row_setup(const EventConsts& e, int iy, int h, int col_lo, int col_hi,
                                               const DevParams& p) {
    RowConsts r;
    float y = fmaf((float)iy, p.px, p.y0);
    float dy = y - e.y_t;
    float c2 = p.c2k * e.sec2 * dy * dy;
    float rem = 9.f - c2;                                  // row chord: c1 u^2 <= 9 - c2
    float hw = sqrt_approx(fmaxf(rem, 0.f) * p.half_sz2);
    float zc = fmaf(e.t, dy, e.z_t);                       // u = 0 on the line z = z~ + t dy
    int lo = max(col_lo, __float2int_ru((zc - hw - p.z0) * p.inv_px));
    int hi = min(col_hi, __float2int_rd((zc + hw - p.z0) * p.inv_px));
    int len = rem >= 0.f ? max(0, hi - lo + 1) : 0;
    if (NH > 1) {
        int part = (len + NH - 1) / NH;
        int first = min(len, h * part);
        len = min(len - first, part);
        lo += first;
    }
    float ysec = y * e.sec2;
    float alpha = p.ak * ysec;
    r.u0 = fmaf((float)lo, p.px, p.z0) - zc;
    r.c2s = -kLH * c2;
    r.betas = kSqrtLH * p.bk * ysec * e.t * dy;
    r.delta = p.d1k * e.sec2 * e.sec2 * fmaf(y, y, p.R2) + p.d2k * ysec * e.t * e.t * y
              + p.d3k * ysec * fmaf(2.f * e.t, e.t, 1.f) * dy;
    if (p.gB != 0.f) {                                     // Eq. 12 with gamma != 0
        const float sec3 = e.sec2 * e.sec2 * rsqrt_approx(e.sec2);
        r.betas -= kSqrtLH * p.gB * sec3 * dy;
        r.delta -= sec3 * e.t * fmaf(p.gD0, y, 2.f * p.gB * dy);
    }
    r.alphas = kSqrtLH * alpha;
    r.eps = 2.f * e.t * alpha;
    r.lo = lo;
    r.len = len;
    return r;
}

// P (up to the constant K) at pixel j of the row part.
__device__ __forceinline__ float kernel_value(const RowConsts& r, float jf, float px, float c1s) {
    float u = fmaf(jf, px, r.u0);
    float e2 = fmaf(c1s * u, u, r.c2s);
    float ba = fmaf(r.alphas, u, r.betas);
    float D = fmaf(r.eps, u, r.delta);
    float rs = rsqrt_approx(D);
    float bar = ba * rs;
    e2 = fmaf(bar, bar, e2);
    return rs * ex2_approx(e2);
}

// ------------------------------------------------------------------------------------------------------
// Binning: sub-tile of the event's reconstructed point; NB = nby*nbz is the "direct" bin (events that do
// not fit a region: non-finite, |tan theta~| > t_max, or centred outside the halo-extended image).
__device__ __forceinline__ int event_bin(float zu, float zd, float dl, const DevParams& p) {
    EventConsts e = event_setup(zu, zd, dl, p);
    float fz = (e.z_t - p.z0) * p.inv_px;
    bool regular = e.finite && fabsf(e.t) <= p.t_max && e.fy >= (float)(1 - p.Hy) && e.fy < (float)(p.n_y + p.Hy - 1) &&
                   fz >= (float)(1 - p.Hz) && fz < (float)(p.n_z + p.Hz - 1);
    if (p.nr_max > 0) {                // the row count of the whole ellipse must be one the task table knows
        const int nr = __float2int_rd(e.fy + e.hy_px) - __float2int_ru(e.fy - e.hy_px) + 1;
        regular = regular && nr >= p.nr_min && nr <= p.nr_max;
    }
    if (!regular) return p.nby * p.nbz;
    int iyc = __float2int_rd(e.fy + 0.5f), izc = __float2int_rd(fz + 0.5f);
    int by = (iyc + p.Hy) / p.Sy, bz = (izc + p.Hz) / p.Sz;
    by = min(max(by, 0), p.nby - 1);
    bz = min(max(bz, 0), p.nbz - 1);
    return by * p.nbz + bz;
}

// Histogram of the bins: per-block shared-memory histogram (when it fits), one global atomic per non-empty bin.
constexpr int kBinBlock = 256, kBinPer = 8, kBinSmemMax = 12288;   // threads, events per thread, max bins in smem

__global__ void __launch_bounds__(kBinBlock)
bin_count_kernel(const float* __restrict__ events, int n, const __grid_constant__ DevParams p, int* __restrict__ bin_of,
                 int* __restrict__ counts, int nb1, int use_smem) {
    pdl_wait();
    extern __shared__ int hist[];
    const int tid = threadIdx.x;
    if (use_smem) {
        for (int b = tid; b < nb1; b += kBinBlock) hist[b] = 0;
        __syncthreads();
    }
    const int base = blockIdx.x * (kBinBlock * kBinPer);
#pragma unroll
    for (int q = 0; q < kBinPer; ++q) {
        const int i = base + q * kBinBlock + tid;
        if (i < n) {
            const int b = event_bin(__ldg(events + 3 * (size_t)i), __ldg(events + 3 * (size_t)i + 1), __ldg(events + 3 * (size_t)i + 2), p);
            bin_of[i] = b;
            atomicAdd(use_smem ? hist + b : counts + b, 1);
        }
    }
    if (use_smem) {
        __syncthreads();
        for (int b = tid; b < nb1; b += kBinBlock) {
            const int c = hist[b];
            if (c) atomicAdd(counts + b, c);
        }
    }
}

// One block: exclusive prefix of counts -> starts (and cursors), work items for the regular bins.  Full items
// (chunk events) come first in the list, the partly filled last item of every bin after them, so that the persistent
// event kernel ends on small items.
// meta[0] = number of items, meta[1] = start of the direct bin, meta[2] = its count, meta[3] = work counter (zeroed)
__global__ void bin_scan_kernel(int* __restrict__ counts, int* __restrict__ cursors, WorkItem* __restrict__ items,
                                int* __restrict__ meta, int nb, int chunk) {
    pdl_wait();
    __shared__ int s_ev[1024], s_it[1024], s_pt[1024];
    const int tid = threadIdx.x, T = blockDim.x;
    const int per = (nb + 1 + T - 1) / T;                  // bins per thread, contiguous
    const int b0 = tid * per, b1 = min(nb + 1, b0 + per);
    int ev = 0, it = 0, pt = 0;
    for (int b = b0; b < b1; ++b) {
        int c = counts[b];
        ev += c;
        if (b < nb) { it += c / chunk; pt += (c % chunk) != 0; }
    }
    s_ev[tid] = ev; s_it[tid] = it; s_pt[tid] = pt;
    __syncthreads();
    for (int d = 1; d < T; d <<= 1) {                      // Hillis-Steele inclusive scan
        int a = tid >= d ? s_ev[tid - d] : 0, c = tid >= d ? s_it[tid - d] : 0, e = tid >= d ? s_pt[tid - d] : 0;
        __syncthreads();
        s_ev[tid] += a; s_it[tid] += c; s_pt[tid] += e;
        __syncthreads();
    }
    const int n_full = s_it[T - 1];
    int ev_off = s_ev[tid] - ev, it_off = s_it[tid] - it, pt_off = n_full + s_pt[tid] - pt;
    for (int b = b0; b < b1; ++b) {
        int c = counts[b];
        counts[b] = 0;                                     // ready for the next batch (no memset between batches)
        cursors[b] = ev_off;
        if (b < nb) {
            int k = 0;
            for (; k + chunk <= c; k += chunk) items[it_off++] = WorkItem{b, ev_off + k, chunk};
            if (k < c) items[pt_off++] = WorkItem{b, ev_off + k, c - k};
        } else {
            meta[1] = ev_off;
            meta[2] = c;
        }
        ev_off += c;
    }
    if (tid == T - 1) { meta[0] = s_it[tid] + s_pt[tid]; meta[3] = 0; }
}

// Scatter into bin order: ranks inside the block from a shared-memory histogram, one global cursor atomic per
// non-empty bin and block.  (The order of events inside a bin depends on block scheduling; sums are fp32.)
__global__ void __launch_bounds__(kBinBlock)
bin_scatter_kernel(const float* __restrict__ events, int n, const int* __restrict__ bin_of, int* __restrict__ cursors,
                   float* __restrict__ sorted, int nb1, int use_smem) {
    pdl_wait();
    extern __shared__ int hist[];
    const int tid = threadIdx.x;
    const int base = blockIdx.x * (kBinBlock * kBinPer);
    int bin[kBinPer], rank[kBinPer];
    if (use_smem) {
        for (int b = tid; b < nb1; b += kBinBlock) hist[b] = 0;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < kBinPer; ++q) {
            const int i = base + q * kBinBlock + tid;
            bin[q] = i < n ? bin_of[i] : -1;
            rank[q] = bin[q] >= 0 ? atomicAdd(hist + bin[q], 1) : 0;
        }
        __syncthreads();
        for (int b = tid; b < nb1; b += kBinBlock) {
            const int c = hist[b];
            if (c) hist[b] = atomicAdd(cursors + b, c);       // count -> base of this block's run in bin b
        }
        __syncthreads();
    }
#pragma unroll
    for (int q = 0; q < kBinPer; ++q) {
        const int i = base + q * kBinBlock + tid;
        if (i >= n) continue;
        int pos;
        if (use_smem) pos = hist[bin[q]] + rank[q];
        else pos = atomicAdd(cursors + bin_of[i], 1);
        sorted[3 * (size_t)pos] = __ldg(events + 3 * (size_t)i);
        sorted[3 * (size_t)pos + 1] = __ldg(events + 3 * (size_t)i + 1);
        sorted[3 * (size_t)pos + 2] = __ldg(events + 3 * (size_t)i + 2);
    }
}

// ------------------------------------------------------------------------------------------------------
// Compile-time loop: f(integral_constant<int, J>) for J in [J0, J1) - gives inline asm its immediates.
template <int J0, int J1, typename F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (J0 < J1) {
        f(std::integral_constant<int, J0>{});
        static_for<J0 + 1, J1>(f);
    }
}

// Shared-memory accessors on 32-bit shared-space addresses with immediate offsets (LDS/STS [R + imm]).
template <int IMM>
__device__ __forceinline__ float lds_imm(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1 + %2];" : "=f"(v) : "r"(addr), "n"(IMM));
    return v;
}
// acc[addr + IMM] += P * inv for lanes with len > J, predicated (no branch)
template <int IMM, int J>
__device__ __forceinline__ void smem_fma_if(uint32_t addr, float P, float inv, int len) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .f32 t;\n\t"
        "setp.gt.s32 p, %3, %4;\n\t"
        "@p ld.shared.f32 t, [%0 + %5];\n\t"
        "@p fma.rn.f32 t, %1, %2, t;\n\t"
        "@p st.shared.f32 [%0 + %5], t;\n\t}"
        ::"r"(addr), "f"(P), "f"(inv), "r"(len), "n"(J), "n"(IMM)
        : "memory");
}

template <int IMM>
__device__ __forceinline__ void smem_fma(uint32_t addr, float P, float inv) {
    asm volatile(
        "{\n\t.reg .f32 t;\n\t"
        "ld.shared.f32 t, [%0 + %3];\n\t"
        "fma.rn.f32 t, %1, %2, t;\n\t"
        "st.shared.f32 [%0 + %3], t;\n\t}"
        ::"r"(addr), "f"(P), "f"(inv), "n"(IMM)
        : "memory");
}

// Packed fp32x2 arithmetic (sm_100: FFMA2 / FMUL2 / FADD2 - two fp32 operations per issue slot).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// Row constants rescaled so that the Gaussian term is -u'^2 with u' = u * sqrt(-c1s) (saves one FMUL per pixel).
struct RowWalk {
    float u0s, c2s, betas, delta, alphas, eps;   // alphas, eps divided by sqrt(-c1s); u0s multiplied by it
    int lo, len;
};

template <int NH>
__device__ __forceinline__ RowWalk row_walk_setup(const EventConsts& e, int iy, int h, int col_lo, int col_hi,
                                                  const DevParams& p) {
    RowConsts r = row_setup<NH>(e, iy, h, col_lo, col_hi, p);
    RowWalk w;
    w.u0s = r.u0 * p.sq;
    w.c2s = r.c2s;
    w.betas = r.betas;
    w.delta = r.delta;
    w.alphas = r.alphas * p.inv_sq;
    w.eps = r.eps * p.inv_sq;
    w.lo = r.lo;
    w.len = r.len;
    return w;
}

__device__ __forceinline__ float kernel_value_scaled(const RowWalk& r, float jf, float pxs) {
    float u = fmaf(jf, pxs, r.u0s);
    float D = fmaf(r.eps, u, r.delta);
    float ba = fmaf(r.alphas, u, r.betas);
    float rs = rsqrt_approx(D);
    float e2 = fmaf(-u, u, r.c2s);
    float bar = ba * rs;
    e2 = fmaf(bar, bar, e2);
    return rs * ex2_approx(e2);
}

// Slot m -> row index, central rows first (c, c+1, c-1, c+2, ...), so that the first warp gets the 32 longest
// chords and the last one the short caps: warp-uniform loop bounds then fit the ellipse better.  Any 32
// consecutive slots map to rows that are distinct modulo 32 (shared-memory banks).  -1: no such row.
__device__ __forceinline__ int centre_first(int m, int nrows) {
    const int c = nrows >> 1;
    const int r = (m & 1) ? c + ((m + 1) >> 1) : c - (m >> 1);
    return (r >= 0 && r < nrows) ? r : -1;
}

template <bool CF>
__device__ __forceinline__ int row_of_slot(int m, int nrows) {
    if (CF) return centre_first(m, nrows);
    return m < nrows ? m : -1;
}

// One event on one CTA, tiled path.  w_addr / a_addr: 32-bit shared addresses of the region origins; pixel
// (iy, iz) lives at base + 4 * ((iz - rz0) * HS + (iy - ry0)).  THREAD <-> ROW (part h of NH).
template <int NW, int NH, int NR, int NJ, int HS, int U, bool CF, bool PK>
__device__ __forceinline__ void process_event_tiled(float zu, float zd, float dl, const DevParams& p, uint32_t w_addr,
                                                    uint32_t a_addr, int ry0, int rz0, int row_lo, int row_hi, int col_lo,
                                                    int col_hi, float* red_s, unsigned long long& my_evals,
                                                    unsigned long long& my_skipped) {
    constexpr int GT = NW * 32;
    constexpr int RT = GT / NH;                 // threads (rows) per pass
    constexpr int NB = (NJ + U - 1) / U;
    const int tid = threadIdx.x, lane = tid & 31;
    const int h = tid / RT, k = tid - h * RT;   // row part and row slot of this thread
    const float pxs = p.px * p.sq;

    const EventConsts e = event_setup(zu, zd, dl, p);
    int iy_lo, nrows;
    event_rows(e, row_lo, row_hi, iy_lo, nrows);

    float preg[NR][NB * U];
    int len[NR], wmax[NR], wmin[NR];
    uint32_t off[NR];
    float denom = 0.f;
    int cnt = 0;
#pragma unroll
    for (int i = 0; i < NR; ++i) {
        const int r = row_of_slot<CF>(k + i * RT, nrows);
        RowWalk rc;
        rc.u0s = 0.f; rc.c2s = 0.f; rc.betas = 0.f; rc.delta = 1.f; rc.alphas = 0.f; rc.eps = 0.f; rc.lo = rz0; rc.len = 0;
        int iy = ry0;
        if (r >= 0) { iy = iy_lo + r; rc = row_walk_setup<NH>(e, iy, h, col_lo, col_hi, p); }
        len[i] = rc.len;
        off[i] = 4u * (uint32_t)((rc.lo - rz0) * HS + (iy - ry0));
        cnt += rc.len;
        wmax[i] = __reduce_max_sync(0xffffffffu, rc.len);
        wmin[i] = __reduce_min_sync(0xffffffffu, rc.len);
        const uint32_t wa = w_addr + off[i];
        if constexpr (!PK) {
        static_for<0, NB>([&](auto bc) {
            constexpr int jb = decltype(bc)::value * U;
            if (jb + U <= wmin[i]) {                             // warp-uniform: every lane owns these pixels
                static_for<0, U>([&](auto jc) {
                    constexpr int j = jb + decltype(jc)::value;
                    const float P = kernel_value_scaled(rc, (float)j, pxs);
                    denom = fmaf(P, lds_imm<4 * j * HS>(wa), denom);
                    preg[i][j] = P;
                });
            } else if (jb < wmax[i]) {                           // warp-uniform: ragged end of the rows
                static_for<0, U>([&](auto jc) {
                    constexpr int j = jb + decltype(jc)::value;
                    float P = kernel_value_scaled(rc, (float)j, pxs);
                    P = j < rc.len ? P : 0.f;                    // lanes past their span contribute nothing; the
                    const float wv = lds_imm<4 * j * HS>(wa);    // read stays inside the (finite) shared arrays
                    denom = fmaf(P, wv, denom);
                    preg[i][j] = P;
                });
            }
        });
        } else {
        // packed form: two adjacent pixels of the row per fp32x2 operation.  Exponent written as
        // c2s + (bar - v)(bar + v) = c2s - v^2 + bar^2 so that no packed negation is needed.
        static_assert(U % 2 == 0, "packed walk needs an even block");
        const f32x2 EPS2 = pack2(rc.eps, rc.eps), DEL2 = pack2(rc.delta, rc.delta), ALP2 = pack2(rc.alphas, rc.alphas),
                    BET2 = pack2(rc.betas, rc.betas), C2S2 = pack2(rc.c2s, rc.c2s), STEP2 = pack2(2.f * pxs, 2.f * pxs);
        f32x2 V2 = pack2(rc.u0s, rc.u0s + pxs), DEN2 = pack2(0.f, 0.f);
        auto pair_step = [&](auto jc, auto maskc) {
            constexpr int j = decltype(jc)::value;
            constexpr bool MASK = decltype(maskc)::value;
            const f32x2 D2 = fma2(EPS2, V2, DEL2), BA2 = fma2(ALP2, V2, BET2);
            float d0, d1;
            unpack2(D2, d0, d1);
            const f32x2 RS2 = pack2(rsqrt_approx(d0), rsqrt_approx(d1));
            const f32x2 BAR2 = mul2(BA2, RS2);
            const f32x2 E2 = fma2(add2(BAR2, V2), sub2(BAR2, V2), C2S2);
            float e0, e1;
            unpack2(E2, e0, e1);
            float x0 = ex2_approx(e0), x1 = ex2_approx(e1);
            if (MASK) {                                           // 2^e -> 0 for lanes past their span
                x0 = j < rc.len ? x0 : 0.f;
                x1 = j + 1 < rc.len ? x1 : 0.f;
            }
            const f32x2 P2 = mul2(RS2, pack2(x0, x1));
            DEN2 = fma2(P2, pack2(lds_imm<4 * j * HS>(wa), lds_imm<4 * (j + 1) * HS>(wa)), DEN2);
            unpack2(P2, preg[i][j], preg[i][j + 1]);
            V2 = add2(V2, STEP2);
        };
        static_for<0, NB>([&](auto bc) {
            constexpr int jb = decltype(bc)::value * U;
            if (jb + U <= wmin[i]) {                             // warp-uniform: every lane owns these pixels
                static_for<0, U / 2>([&](auto jc) {
                    pair_step(std::integral_constant<int, jb + 2 * decltype(jc)::value>{}, std::false_type{});
                });
            } else if (jb < wmax[i]) {                           // warp-uniform: ragged end of the rows
                static_for<0, U / 2>([&](auto jc) {
                    pair_step(std::integral_constant<int, jb + 2 * decltype(jc)::value>{}, std::true_type{});
                });
            }
        });
        float q0, q1;
        unpack2(DEN2, q0, q1);
        denom += q0 + q1;
        }
        for (int j = NB * U; j < rc.len; ++j) {                  // longer than the register cache (not in tuned configs)
            float P = kernel_value_scaled(rc, (float)j, pxs);
            float wv;
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(wv) : "r"(wa + 4u * (uint32_t)(j * HS)));
            denom = fmaf(P, wv, denom);
        }
    }
    for (int m = k + NR * RT; m <= nrows; m += RT) {             // more rows than NR passes (not in tuned configs)
        const int r = row_of_slot<CF>(m, nrows);
        if (r < 0) continue;
        RowWalk rc = row_walk_setup<NH>(e, iy_lo + r, h, col_lo, col_hi, p);
        const uint32_t wa = w_addr + 4u * (uint32_t)((rc.lo - rz0) * HS + (iy_lo + r - ry0));
        cnt += rc.len;
        for (int j = 0; j < rc.len; ++j) {
            float P = kernel_value_scaled(rc, (float)j, pxs);
            float wv;
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(wv) : "r"(wa + 4u * (uint32_t)(j * HS)));
            denom = fmaf(P, wv, denom);
        }
    }
    my_evals += (unsigned long long)cnt;

    // ---- denominator: sum over the CTA -------------------------------------------------------------------
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) denom += __shfl_xor_sync(0xffffffffu, denom, d);
    if (NW > 1) {
        if (lane == 0) red_s[tid >> 5] = denom;
        __syncthreads();
        denom = 0.f;
#pragma unroll
        for (int q = 0; q < NW; ++q) denom += red_s[q];
    } else {
        __syncwarp();
    }

    // ---- back-projection: acc += P / denominator (private region: plain read-modify-write) --------------------
    const bool ok = (denom > 0.f) && (denom < 3.0e38f);
    if (tid == 0 && !ok) my_skipped += 1ull;
    if (!ok) return;
    const float inv = 1.f / denom;
#pragma unroll
    for (int i = 0; i < NR; ++i) {
        const uint32_t aa = a_addr + off[i];
        static_for<0, NB>([&](auto bc) {
            constexpr int jb = decltype(bc)::value * U;
            if (jb + U <= wmin[i]) {
                static_for<0, U>([&](auto jc) {
                    constexpr int j = jb + decltype(jc)::value;
                    smem_fma<4 * j * HS>(aa, preg[i][j], inv);
                });
            } else if (jb < wmax[i]) {
                static_for<0, U>([&](auto jc) {
                    constexpr int j = jb + decltype(jc)::value;
                    smem_fma_if<4 * j * HS, j>(aa, preg[i][j], inv, len[i]);
                });
            }
        });
        if (len[i] > NB * U) {
            const int r = row_of_slot<CF>(k + i * RT, nrows);
            RowWalk rc = row_walk_setup<NH>(e, iy_lo + r, h, col_lo, col_hi, p);
            for (int j = NB * U; j < rc.len; ++j) {
                float v = kernel_value_scaled(rc, (float)j, pxs) * inv, t;
                const uint32_t ad = aa + 4u * (uint32_t)(j * HS);
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(t) : "r"(ad));
                asm volatile("st.shared.f32 [%0], %1;" ::"r"(ad), "f"(t + v) : "memory");
            }
        }
    }
    for (int m = k + NR * RT; m <= nrows; m += RT) {
        const int r = row_of_slot<CF>(m, nrows);
        if (r < 0) continue;
        RowWalk rc = row_walk_setup<NH>(e, iy_lo + r, h, col_lo, col_hi, p);
        const uint32_t aa = a_addr + 4u * (uint32_t)((rc.lo - rz0) * HS + (iy_lo + r - ry0));
        for (int j = 0; j < rc.len; ++j) {
            float v = kernel_value_scaled(rc, (float)j, pxs) * inv, t;
            const uint32_t ad = aa + 4u * (uint32_t)(j * HS);
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(t) : "r"(ad));
            asm volatile("st.shared.f32 [%0], %1;" ::"r"(ad), "f"(t + v) : "memory");
        }
    }
}

// Tiled path: work items (sub-tile, chunk of sorted events), private shared-memory region per CTA.
template <int NW, int NH, int NR, int NJ, int HS, int U, bool CF, int MINB, bool PK>
__global__ void __launch_bounds__(NW * 32, MINB)
mlem_rows_kernel(const float* __restrict__ sorted, const WorkItem* __restrict__ items, int* __restrict__ meta,
                 const __grid_constant__ DevParams p, const float* __restrict__ wT, float* __restrict__ accT,
                 unsigned long long* __restrict__ counters) {
    constexpr int GT = NW * 32;
    extern __shared__ __align__(16) float smem[];
    const int WZ = p.WZ;
    float* w_s = smem;
    float* acc_s = smem + HS * WZ;
    const uint32_t w_addr = (uint32_t)__cvta_generic_to_shared(w_s);
    const uint32_t a_addr = (uint32_t)__cvta_generic_to_shared(acc_s);
    __shared__ float red_s[2][NW];
    __shared__ int item_s;
    const int tid = threadIdx.x;
    const int n_items = meta[0];
    unsigned long long my_evals = 0, my_skipped = 0;
    int parity = 0;

    while (true) {
        if (tid == 0) item_s = atomicAdd(meta + 3, 1);
        __syncthreads();
        const int item = item_s;
        if (item >= n_items) break;
        const WorkItem wi = items[item];
        const int by = wi.bin / p.nbz, bz = wi.bin - by * p.nbz;
        const int ry0 = by * p.Sy - 2 * p.Hy, rz0 = bz * p.Sz - 2 * p.Hz;        // region origin (pixel indices)
        const int row_lo = max(0, ry0), row_hi = min(p.n_y - 1, ry0 + p.Sy + 2 * p.Hy - 1);
        const int col_lo = max(0, rz0), col_hi = min(p.n_z - 1, rz0 + WZ - 1);
        // stage w (several loads in flight per thread), zero the accumulator region
        for (int i0 = tid; i0 < HS * WZ; i0 += 4 * GT) {
            float v[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = i0 + q * GT;
                const int c = i / HS, r = i - c * HS;
                const int iz = rz0 + c, iy = ry0 + r;
                v[q] = 0.f;
                if (i < HS * WZ && iz >= col_lo && iz <= col_hi && iy >= row_lo && iy <= row_hi)
                    v[q] = __ldg(wT + (size_t)iz * p.n_y + iy);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = i0 + q * GT;
                if (i < HS * WZ) { w_s[i] = v[q]; acc_s[i] = 0.f; }
            }
        }
        __syncthreads();
        const float* ev = sorted + 3 * (size_t)wi.start;
        float zu = __ldg(ev), zd = __ldg(ev + 1), dl = __ldg(ev + 2);
        for (int q = 0; q < wi.count; ++q) {
            float nzu = 0.f, nzd = 0.f, ndl = 0.f;
            if (q + 1 < wi.count) { nzu = __ldg(ev + 3 * (q + 1)); nzd = __ldg(ev + 3 * (q + 1) + 1); ndl = __ldg(ev + 3 * (q + 1) + 2); }
            process_event_tiled<NW, NH, NR, NJ, HS, U, CF, PK>(zu, zd, dl, p, w_addr, a_addr, ry0, rz0, row_lo, row_hi, col_lo, col_hi,
                                                    red_s[parity], my_evals, my_skipped);
            parity ^= 1;
            zu = nzu; zd = nzd; dl = ndl;
        }
        __syncthreads();
        // flush the private region into the global transposed accumulator
        for (int i = tid; i < HS * WZ; i += GT) {
            const int c = i / HS, r = i - c * HS;
            const int iz = rz0 + c, iy = ry0 + r;
            const float v = acc_s[i];
            if (v != 0.f && iz >= col_lo && iz <= col_hi && iy >= row_lo && iy <= row_hi)
                red_add_f32(accT + (size_t)iz * p.n_y + iy, v);
        }
        __syncthreads();
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) my_evals += __shfl_xor_sync(0xffffffffu, my_evals, d);
    if ((tid & 31) == 0 && my_evals) atomicAdd(counters + 0, my_evals);
    if (tid == 0 && my_skipped) atomicAdd(counters + 1, my_skipped);
}

// Direct path: events of the "direct" bin (rare: non-finite, extreme angles, far outside the image), or every
// event when a region does not fit shared memory.  One warp per event, thread <-> row, w read from the global
// transposed image, back-projection with red.global.add.f32, P recomputed in the second pass.  Simple on purpose.
__global__ void __launch_bounds__(128)
mlem_rows_direct_kernel(const float* __restrict__ sorted, int stride, int* __restrict__ meta,
                        const __grid_constant__ DevParams p, const float* __restrict__ wT, float* __restrict__ accT,
                        unsigned long long* __restrict__ counters) {
    pdl_wait();
    const int lane = threadIdx.x & 31;
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
    const int start = meta[1], count = meta[2];
    unsigned long long my_evals = 0, my_skipped = 0;
    for (int q = warp; q < count; q += n_warps) {
        const float* ev = sorted + (size_t)stride * (size_t)(start + q);      // raw triple at the head of the slot
        const EventConsts e = event_setup(__ldg(ev), __ldg(ev + 1), __ldg(ev + 2), p);
        int iy_lo, nrows;
        event_rows(e, 0, p.n_y - 1, iy_lo, nrows);
        float denom = 0.f;
        for (int r = lane; r < nrows; r += 32) {
            const RowConsts rc = row_setup<1>(e, iy_lo + r, 0, 0, p.n_z - 1, p);
            const float* wp = wT + (size_t)rc.lo * p.n_y + (iy_lo + r);
            my_evals += (unsigned long long)rc.len;
            for (int j = 0; j < rc.len; ++j) denom = fmaf(kernel_value(rc, (float)j, p.px, p.c1s), __ldg(wp + (size_t)j * p.n_y), denom);
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) denom += __shfl_xor_sync(0xffffffffu, denom, d);
        const bool ok = (denom > 0.f) && (denom < 3.0e38f);
        if (lane == 0 && !ok) my_skipped += 1ull;
        if (!ok) continue;
        const float inv = 1.f / denom;
        for (int r = lane; r < nrows; r += 32) {
            const RowConsts rc = row_setup<1>(e, iy_lo + r, 0, 0, p.n_z - 1, p);
            float* ap = accT + (size_t)rc.lo * p.n_y + (iy_lo + r);
            for (int j = 0; j < rc.len; ++j) red_add_f32(ap + (size_t)j * p.n_y, kernel_value(rc, (float)j, p.px, p.c1s) * inv);
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) my_evals += __shfl_xor_sync(0xffffffffu, my_evals, d);
    if (lane == 0 && my_evals) atomicAdd(counters + 0, my_evals);
    if (lane == 0 && my_skipped) atomicAdd(counters + 1, my_skipped);
    // this kernel always follows the tiled event kernel in the stream: reset the work counter for the next run over
    // the same sorted events (jpet_reconstruct sorts once and iterates)
    if (blockIdx.x == 0 && threadIdx.x == 0) meta[3] = 0;
}

// |E_j| only (jpet_count_evals): thread per event, rows in a loop, no kernel values.
__global__ void count_evals_kernel(const float* __restrict__ events, long long n, const __grid_constant__ DevParams p,
                                   unsigned long long* __restrict__ counters) {
    unsigned long long evals = 0, skipped = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        EventConsts e = event_setup(events[3 * i], events[3 * i + 1], events[3 * i + 2], p);
        int iy_lo, nrows, cnt = 0;
        event_rows(e, 0, p.n_y - 1, iy_lo, nrows);
        for (int r = 0; r < nrows; ++r) cnt += row_setup<1>(e, iy_lo + r, 0, 0, p.n_z - 1, p).len;
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
