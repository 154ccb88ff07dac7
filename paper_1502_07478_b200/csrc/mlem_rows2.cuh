// mlem_rows2.cuh - second-generation event kernel of the list-mode MLEM hot path (sm_100a).
//
// Same mathematics and the same tiling as mlem_rows_kernel (mlem_kernels.cuh: events sorted by image sub-tile,
// private shared-memory w / accumulator regions per CTA, THREAD <-> ELLIPSE ROW, kernel values cached in
// registers between the denominator pass and the back-projection pass).  What changes is the instruction
// count per event, which ncu showed to be the bound (issue slots 77 % busy, 50 thread-instructions per kernel
// evaluation against 10 algorithmic):
//
//   * the per-event part of step 1 - Eq. 2 and everything of Eq. 7-10 / B.3
//      that does not depend on the pixel - is evaluated ONCE per event by the
//     binning pass and stored with the sorted event as a 64-byte record (EventRec).  Along the ellipse all
//     row constants are polynomials in dy = y - y~ (y = y~ + dy):
//         c2s    = K2 dy^2                       betas = dy (B1 + KB dy)
//         alphas = A0 + A1 dy                    eps   = E0 + E1 dy
//         delta  = D0 + dy (D1 + D2 dy)
//         half chord^2 [pixels^2] = H0p + H2p dy^2      chord centre [pixels] = Z0 + T1 dy
//     so a row costs about 25 instructions instead of 61 and the warp no longer repeats Eq. 2;
//   * rows are dealt to lanes so that a warp's rows have nearly equal chords: the central 32*NA rows go to
//     the "A" warps (warp 0 the central 32, warp b 16 rows on either side of block b-1; NH > 1 splits every
//     row in NH parts that live in DIFFERENT warps, so that no two lanes of a warp share a bank), the
//     remaining cap rows go to one "B" warp that splits the longer ones in 2 or 4 parts to fill its lanes;
//   * per-event bookkeeping is 32-bit and flushed once per work item.
//
// Citations are /root/reference/PAPER.md lines.  Nothing here is shared with oracle/.
#pragma once
#include "mlem_kernels.cuh"

namespace jpet {

// Per-event constants, written by bin_scatter_rec_kernel, read (broadcast) by mlem_rows2_kernel.
struct __align__(16) EventRec {
    float yoff, K2, B1, KB;      // dy = iy * px + yoff;  c2s = K2 dy^2;  betas = dy (B1 + KB dy)
    float A0, A1, E0, E1;        // alphas = A0 + A1 dy;  eps = E0 + E1 dy
    float D0, D1, D2, H2p;       // delta = D0 + dy (D1 + D2 dy);  hw^2 = H0p + H2p dy^2  (pixels^2)
    float Z0, T1;                // chord centre = Z0 + T1 dy  (pixels, column 0 = 0)
    int iy_lo, nrows;            // rows of the ellipse clipped to the grid
};
static_assert(sizeof(EventRec) == 64, "EventRec must be 64 bytes");

// Eq. 2 and the per-event factors of Eq. 7-10 / B.3 (see the header of mlem_kernels.cuh for the algebra).
__device__ __forceinline__ EventRec make_event_rec(float zu, float zd, float dl, const DevParams& p) {
    const EventConsts e = event_setup(zu, zd, dl, p);
    EventRec r;
    const float t = e.t, sec2 = e.sec2, yt = e.y_t;
    r.yoff = p.y0 - yt;
    r.K2 = -kLH * p.c2k * sec2;
    r.KB = kSqrtLH * p.bk * sec2 * t;
    r.B1 = r.KB * yt;
    r.A1 = kSqrtLH * p.ak * sec2 * p.inv_sq;
    r.A0 = r.A1 * yt;
    r.E1 = 2.f * t * p.ak * sec2 * p.inv_sq;
    r.E0 = r.E1 * yt;
    const float s4 = sec2 * sec2, st2 = sec2 * t * t;
    const float G1 = fmaf(p.d2k, st2, p.d1k * s4);
    const float G2 = p.d3k * fmaf(2.f, st2, sec2);
    r.D0 = fmaf(G1, yt * yt, p.d1k * s4 * p.R2);
    r.D1 = fmaf(2.f, G1, G2) * yt;
    r.D2 = G1 + G2;
    if (p.gB != 0.f) {                                     // Eq. 12 with gamma != 0 (DevParams, mlem_kernels.cuh)
        const float sec3 = sec2 * sec2 * rsqrt_approx(sec2);
        const float G3 = sec3 * t;
        r.B1 -= kSqrtLH * p.gB * sec3;
        r.D0 -= p.gD0 * G3 * yt;
        r.D1 -= (p.gD0 + 2.f * p.gB) * G3;
    }
    r.H2p = -p.c2k * sec2 * p.half_sz2 * p.inv_px * p.inv_px;
    r.Z0 = (e.z_t - p.z0) * p.inv_px;
    r.T1 = t * p.inv_px;
    int iy_lo, nrows;
    if (p.nr_max > 0) event_rows(e, -(1 << 24), 1 << 24, iy_lo, nrows);     // whole ellipse (mlem_rows3.cuh clips per row)
    else event_rows(e, 0, p.n_y - 1, iy_lo, nrows);
    r.iy_lo = iy_lo;
    r.nrows = nrows;
    return r;
}

// Scatter into bin order, as bin_scatter_kernel, but the regular bins receive EventRec records; the events
// of the direct bin keep their raw triple in the first three floats of their 64-byte slot.
__global__ void __launch_bounds__(kBinBlock)
bin_scatter_rec_kernel(const float* __restrict__ events, int n, const int* __restrict__ bin_of, int* __restrict__ cursors,
                       EventRec* __restrict__ sorted, const __grid_constant__ DevParams p, int nb1, int use_smem) {
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
            if (c) hist[b] = atomicAdd(cursors + b, c);
        }
        __syncthreads();
    }
#pragma unroll
    for (int q = 0; q < kBinPer; ++q) {
        const int i = base + q * kBinBlock + tid;
        if (i >= n) continue;
        int pos, b;
        if (use_smem) { b = bin[q]; pos = hist[b] + rank[q]; }
        else { b = bin_of[i]; pos = atomicAdd(cursors + b, 1); }
        const float zu = __ldg(events + 3 * (size_t)i), zd = __ldg(events + 3 * (size_t)i + 1), dl = __ldg(events + 3 * (size_t)i + 2);
        float4* dst = reinterpret_cast<float4*>(sorted + pos);
        if (b == nb1 - 1) {
            dst[0] = make_float4(zu, zd, dl, 0.f);
        } else {
            const EventRec r = make_event_rec(zu, zd, dl, p);
            dst[0] = make_float4(r.yoff, r.K2, r.B1, r.KB);
            dst[1] = make_float4(r.A0, r.A1, r.E0, r.E1);
            dst[2] = make_float4(r.D0, r.D1, r.D2, r.H2p);
            dst[3] = make_float4(r.Z0, r.T1, __int_as_float(r.iy_lo), __int_as_float(r.nrows));
        }
    }
}

// One event on one CTA.  Warp roles and the lane <-> row map are described in the header.
template <int NA, int NH, int NBW, int NJ, int HS, int U, bool PK>
__device__ __forceinline__ void process_event_rows2(const float4 r0, const float4 r1, const float4 r2, const float4 r3,
                                                    const DevParams& p, uint32_t w_addr, uint32_t a_addr, int ry0, int rz0,
                                                    int col_lo, int col_hi, float* red_s, int& my_evals, int& my_skipped) {
    constexpr int NW = NA * NH + NBW;
    constexpr int NB = (NJ + U - 1) / U;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float pxs = p.pxs;
    const int iy_lo = __float_as_int(r3.z), nrows = __float_as_int(r3.w);
    const int iy_hi = iy_lo + nrows - 1;

    // ---- lane -> (row, part of the row) -----------------------------------------------------------------------
    // central block of 32*NA rows starts at iyA_lo; when there are more rows, the extra ones (caps) lie
    // ceil(ncap/2) below and floor(ncap/2) above it.
    const int ncap = max(0, nrows - 32 * NA);
    const int iyC0 = iy_lo + ((nrows - 32 * NA + 1) >> 1) + 16 * (NA - 1);      // first row of the central 32
    int iy, part = 0, sh = 0;
    bool valid;
    if (NBW == 0 || warp < NA * NH) {
        const int blk = (NA > 1) ? warp % NA : 0;
        iy = iyC0 + lane + ((lane < 16) ? -16 * blk : 16 * blk);
        valid = (iy >= iy_lo) && (iy <= iy_hi);
        if (NH > 1) { part = warp / NA; sh = (NH == 2) ? 1 : 2; }
    } else {
        // cap rows c = 0, 1, ...: alternately below and above the central block (chords decrease with c);
        // s: every cap row gets 2^s parts; the first nx rows get twice as many to use the lanes left over
        int s = ncap <= 8 ? 2 : (ncap <= 16 ? 1 : 0);
        int nx = (s == 2) ? 0 : ((32 >> s) - ncap);
        const int Lx = nx << (s + 1);
        int c;
        if (lane < Lx) { sh = s + 1; c = lane >> sh; part = lane & ((1 << sh) - 1); }
        else { const int l2 = lane - Lx; sh = s; c = nx + (l2 >> s); part = l2 & ((1 << s) - 1); }
        const int iyA_lo = iyC0 - 16 * (NA - 1), iyA_hi = iyC0 + 31 + 16 * (NA - 1);
        iy = (c & 1) ? iyA_hi + 1 + (c >> 1) : iyA_lo - 1 - (c >> 1);
        valid = c < ncap;
    }

    // ---- row constants (polynomials in dy) and the row's span ---------------------------------------------------
    RowWalk rc;
    {
        const float dy = fmaf((float)iy, p.px, r0.x);
        const float dy2 = dy * dy;
        rc.c2s = r0.y * dy2;
        rc.betas = dy * fmaf(r0.w, dy, r0.z);
        rc.alphas = fmaf(r1.y, dy, r1.x);
        rc.eps = fmaf(r1.w, dy, r1.z);
        rc.delta = fmaf(dy, fmaf(r2.z, dy, r2.y), r2.x);
        const float hw2 = fmaf(r2.w, dy2, p.H0p);
        const float hw = sqrt_approx(fmaxf(hw2, 0.f));
        const float zcp = fmaf(r3.y, dy, r3.x);
        int lo = max(col_lo, __float2int_ru(zcp - hw));
        const int hi = min(col_hi, __float2int_rd(zcp + hw));
        int len = (valid && hw2 >= 0.f) ? max(0, hi - lo + 1) : 0;
        if (NH > 1 || NBW > 0) {
            const int plen = (len + (1 << sh) - 1) >> sh;
            const int first = min(len, part * plen);
            len = min(len - first, plen);
            lo += first;
        }
        if (len == 0) { lo = rz0; iy = ry0; rc.delta = 1.f; rc.eps = 0.f; }     // keep idle lanes inside the region
        rc.u0s = ((float)lo - zcp) * pxs;
        rc.lo = lo;
        rc.len = len;
    }
    const uint32_t off = 4u * (uint32_t)((rc.lo - rz0) * HS + (iy - ry0));
    const int wmax = __reduce_max_sync(0xffffffffu, rc.len);
    const int wmin = __reduce_min_sync(0xffffffffu, rc.len);
    my_evals += rc.len;

    // ---- pass 1: kernel values (Eq. 7) into registers, denominator -----------------------------------------------
    float preg[NB * U];
    float denom = 0.f;
    const uint32_t wa = w_addr + off;
    if constexpr (!PK) {
        static_for<0, NB>([&](auto bc) {
            constexpr int jb = decltype(bc)::value * U;
            if (jb + U <= wmin) {
                static_for<0, U>([&](auto jc) {
                    constexpr int j = jb + decltype(jc)::value;
                    const float P = kernel_value_scaled(rc, (float)j, pxs);
                    denom = fmaf(P, lds_imm<4 * j * HS>(wa), denom);
                    preg[j] = P;
                });
            } else if (jb < wmax) {
                static_for<0, U>([&](auto jc) {
                    constexpr int j = jb + decltype(jc)::value;
                    float P = kernel_value_scaled(rc, (float)j, pxs);
                    P = j < rc.len ? P : 0.f;
                    denom = fmaf(P, lds_imm<4 * j * HS>(wa), denom);
                    preg[j] = P;
                });
            }
        });
    } else {
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
            if (MASK) {
                x0 = j < rc.len ? x0 : 0.f;
                x1 = j + 1 < rc.len ? x1 : 0.f;
            }
            const f32x2 P2 = mul2(RS2, pack2(x0, x1));
            DEN2 = fma2(P2, pack2(lds_imm<4 * j * HS>(wa), lds_imm<4 * (j + 1) * HS>(wa)), DEN2);
            unpack2(P2, preg[j], preg[j + 1]);
            V2 = add2(V2, STEP2);
        };
        static_for<0, NB>([&](auto bc) {
            constexpr int jb = decltype(bc)::value * U;
            if (jb + U <= wmin) {
                static_for<0, U / 2>([&](auto jc) {
                    pair_step(std::integral_constant<int, jb + 2 * decltype(jc)::value>{}, std::false_type{});
                });
            } else if (jb < wmax) {
                static_for<0, U / 2>([&](auto jc) {
                    pair_step(std::integral_constant<int, jb + 2 * decltype(jc)::value>{}, std::true_type{});
                });
            }
        });
        float q0, q1;
        unpack2(DEN2, q0, q1);
        denom = q0 + q1;
    }

    // ---- denominator: sum over the CTA --------------------------------------------------------------------------
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) denom += __shfl_xor_sync(0xffffffffu, denom, d);
    if (NW > 1) {
        if (lane == 0) red_s[warp] = denom;
        __syncthreads();
        denom = 0.f;
#pragma unroll
        for (int q = 0; q < NW; ++q) denom += red_s[q];
    } else {
        __syncwarp();
    }
    const bool ok = (denom > 0.f) && (denom < 3.0e38f);
    if (!ok) { if (tid == 0) my_skipped += 1; return; }
    const float inv = 1.f / denom;

    // ---- pass 2: acc += P / denominator (private region, one owner lane per pixel: plain read-modify-write) -------
    const uint32_t aa = a_addr + off;
    static_for<0, NB>([&](auto bc) {
        constexpr int jb = decltype(bc)::value * U;
        if (jb + U <= wmin) {
            static_for<0, U>([&](auto jc) {
                constexpr int j = jb + decltype(jc)::value;
                smem_fma<4 * j * HS>(aa, preg[j], inv);
            });
        } else if (jb < wmax) {
            static_for<0, U>([&](auto jc) {
                constexpr int j = jb + decltype(jc)::value;
                smem_fma_if<4 * j * HS, j>(aa, preg[j], inv, rc.len);
            });
        }
    });
}

template <int NA, int NH, int NBW, int NJ, int HS, int U, bool PK, int MINB>
__global__ void __launch_bounds__((NA * NH + NBW) * 32, MINB)
mlem_rows2_kernel(const EventRec* __restrict__ sorted, const WorkItem* __restrict__ items, int* __restrict__ meta,
                  const __grid_constant__ DevParams p, const float* __restrict__ wT, float* __restrict__ accT,
                  unsigned long long* __restrict__ counters) {
    constexpr int NW = NA * NH + NBW;
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
    int my_evals = 0, my_skipped = 0;
    unsigned long long tot_evals = 0;
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
        const float4* rec = reinterpret_cast<const float4*>(sorted + wi.start);
        float4 r0 = __ldg(rec), r1 = __ldg(rec + 1), r2 = __ldg(rec + 2), r3 = __ldg(rec + 3);
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
        for (int q = 0; q < wi.count; ++q) {
            float4 n0 = r0, n1 = r1, n2 = r2, n3 = r3;
            if (q + 1 < wi.count) {
                const float4* nx = rec + 4 * (q + 1);
                n0 = __ldg(nx); n1 = __ldg(nx + 1); n2 = __ldg(nx + 2); n3 = __ldg(nx + 3);
            }
            process_event_rows2<NA, NH, NBW, NJ, HS, U, PK>(r0, r1, r2, r3, p, w_addr, a_addr, ry0, rz0, col_lo, col_hi,
                                                            red_s[parity], my_evals, my_skipped);
            parity ^= 1;
            r0 = n0; r1 = n1; r2 = n2; r3 = n3;
        }
        tot_evals += (unsigned long long)my_evals;
        my_evals = 0;
        __syncthreads();
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
    for (int d = 16; d > 0; d >>= 1) tot_evals += __shfl_xor_sync(0xffffffffu, tot_evals, d);
    if ((tid & 31) == 0 && tot_evals) atomicAdd(counters + 0, tot_evals);
    if (tid == 0 && my_skipped) atomicAdd(counters + 1, (unsigned long long)my_skipped);
}

}  // namespace jpet
