// sort_kernels.cuh - counting sort of the events by image sub-tile and the work-item list of the tiled event kernel.
//
//   bin_count_kernel        Eq. 2 per event -> sub-tile of (y~, z~) and the ellipse's row range
//                           (event_place, common.cuh); histogram of the bins
//   bin_scan_kernel         exclusive prefix of the histogram; work items (sub-tile, chunk of sorted events)
//   bin_scatter_rec_kernel  the 64-byte record of every event (make_event_rec) written in bin order
//
// Events are read ONCE per kernel with coalesced 16-byte loads into a shared-memory tile (12 bytes per event, so a
// thread's own triple is not a vector; the block's 2048 events are 1536 aligned float4); a block whose events do not
// start on a 16-byte boundary (a caller's slice at an odd offset) takes scalar loads.
#pragma once
#include "common.cuh"

namespace jpet {

// Where an event goes in the sort, decided ONCE per event (bin_count_kernel) and carried to the scatter pass in one
// word: the bin (sub-tile of the reconstructed point, + nby * nbz for the events of degree class 1; n_cls * nby * nbz =
// the "direct" bin for events that do not fit a region:
// non-finite, |tan theta~| > t_max, centred outside the halo-extended image, or a row count the task table does not
// hold) and the row range of the ellipse.  Not inlined: both sort kernels execute the same instructions, so the row
// count that admitted an event to a regular bin is the one its record carries.
struct Place { int bin, rows; };

static __device__ __noinline__ Place event_place(float zu, float zd, float dl, const DevParams& p) {
    const EventConsts e = event_setup(zu, zd, dl, p);
    const float fz = (e.z_t - p.z0) * p.inv_px;
    bool regular = e.finite && fabsf(e.t) <= p.t_max && e.fy >= (float)(1 - p.Hy) && e.fy < (float)(p.n_y + p.Hy - 1) &&
                   fz >= (float)(1 - p.Hz) && fz < (float)(p.n_z + p.Hz - 1);
    int iy_lo, nrows;
    if (p.nr_max > 0) event_rows(e, -(1 << 22), 1 << 22, iy_lo, nrows);     // whole ellipse (mlem_rows.cuh clips per row)
    else event_rows(e, 0, p.n_y - 1, iy_lo, nrows);
    if (p.nr_max > 0) regular = regular && nrows >= p.nr_min && nrows <= p.nr_max;
    Place pl;
    pl.rows = pack_rows(iy_lo, min(nrows, 255));
    const int nb = p.nby * p.nbz;
    pl.bin = nb * p.n_cls;
    if (regular) {
        const int iyc = __float2int_rd(e.fy + 0.5f), izc = __float2int_rd(fz + 0.5f);
        const int by = min(max((iyc + p.Hy) / p.Sy, 0), p.nby - 1), bz = min(max((izc + p.Hz) / p.Sz, 0), p.nbz - 1);
        pl.bin = by * p.nbz + bz;
        if (p.n_cls == 2 && low_degree_ok(e, p)) pl.bin += nb;       // degree class 1: the degree-3 instance
    }
    return pl;
}

constexpr int kBinBlock = 256, kBinPer = 8, kBinSmemMax = 12288;   // threads, events per thread, max bins in smem
constexpr int kBinTile = kBinBlock * kBinPer;                       // events per block

// events [base, base + kBinTile) -> tile[3 * kBinTile] (floats), zero-filled past n.
__device__ __forceinline__ void load_event_tile(const float* __restrict__ events, int n, int base, float* tile) {
    const int tid = threadIdx.x;
    const int cnt = min(kBinTile, n - base);
    const float* src = events + 3 * (size_t)base;
    const int nf = 3 * cnt;
    if ((reinterpret_cast<uintptr_t>(src) & 15u) == 0) {
        const float4* src4 = reinterpret_cast<const float4*>(src);
        float4* dst4 = reinterpret_cast<float4*>(tile);
        const int n4 = nf >> 2;
#pragma unroll
        for (int q = 0; q < (3 * kBinTile / 4 + kBinBlock - 1) / kBinBlock; ++q) {
            const int i = q * kBinBlock + tid;
            if (i < n4) dst4[i] = __ldg(src4 + i);
        }
        for (int i = 4 * n4 + tid; i < nf; i += kBinBlock) tile[i] = __ldg(src + i);
    } else {
        for (int i = tid; i < nf; i += kBinBlock) tile[i] = __ldg(src + i);
    }
}

// Histogram of the bins: per-block shared-memory histogram (when it fits), one global atomic per non-empty bin.
// place[i] = (bin, packed row range) of event i.
__global__ void __launch_bounds__(kBinBlock)
bin_count_kernel(const float* __restrict__ events, int n, const __grid_constant__ DevParams p, int2* __restrict__ place,
                 int* __restrict__ counts, int nb1, int use_smem) {
    pdl_wait();
    extern __shared__ __align__(16) float bin_smem[];
    float* tile = bin_smem;
    int* hist = reinterpret_cast<int*>(bin_smem + 3 * kBinTile);
    const int tid = threadIdx.x;
    const int base = blockIdx.x * kBinTile;
    load_event_tile(events, n, base, tile);
    if (use_smem)
        for (int b = tid; b < nb1; b += kBinBlock) hist[b] = 0;
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kBinPer; ++q) {
        const int k = q * kBinBlock + tid, i = base + k;
        if (i < n) {
            const Place pl = event_place(tile[3 * k], tile[3 * k + 1], tile[3 * k + 2], p);
            place[i] = make_int2(pl.bin, pl.rows);
            atomicAdd(use_smem ? hist + pl.bin : counts + pl.bin, 1);
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
// nb: regular bins of all degree classes, nb0: those of class 0 (the first nb0 bins).  meta: see MetaWord (common.cuh).
__global__ void bin_scan_kernel(int* __restrict__ counts, int* __restrict__ cursors, WorkItem* __restrict__ items,
                                int* __restrict__ meta, int nb, int nb0, int chunk) {
    pdl_wait();
    __shared__ int s_ev[1024], s_it[1024], s_pt[1024];
    __shared__ int s_full0, s_part0;
    const int tid = threadIdx.x, T = blockDim.x;
    if (tid == 0) { s_full0 = 0; s_part0 = 0; }
    __syncthreads();
    const int per = (nb + 1 + T - 1) / T;                  // bins per thread, contiguous
    const int b0 = tid * per, b1 = min(nb + 1, b0 + per);
    int ev = 0, it = 0, pt = 0, it0 = 0, pt0 = 0;
    for (int b = b0; b < b1; ++b) {
        int c = counts[b];
        ev += c;
        if (b < nb) { it += c / chunk; pt += (c % chunk) != 0; }
        if (b < nb0) { it0 += c / chunk; pt0 += (c % chunk) != 0; }
    }
    if (it0) atomicAdd(&s_full0, it0);
    if (pt0) atomicAdd(&s_part0, pt0);
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
            meta[kMetaDirectStart] = ev_off;
            meta[kMetaDirectCount] = c;
        }
        ev_off += c;
    }
    if (tid == T - 1) {
        meta[kMetaItems] = s_it[tid] + s_pt[tid];
        meta[kMetaFull] = n_full;
        meta[kMetaFull0] = s_full0;
        meta[kMetaPart0] = s_part0;
        meta[kMetaCounter0] = 0;
        meta[kMetaCounter1] = 0;
    }
}

// Scatter into bin order: ranks inside the block from a shared-memory histogram, one global cursor atomic per
// non-empty bin and block.  (The order of events inside a bin depends on block scheduling; sums are fp32.)  The
// regular bins receive EventRec records; the events of the direct bin keep their raw triple in the first three floats
// of their 64-byte slot.
__global__ void __launch_bounds__(kBinBlock)
bin_scatter_rec_kernel(const float* __restrict__ events, int n, const int2* __restrict__ place, int* __restrict__ cursors,
                       EventRec* __restrict__ sorted, const __grid_constant__ DevParams p, int nb1, int use_smem) {
    pdl_wait();
    extern __shared__ __align__(16) float bin_smem[];
    float* tile = bin_smem;
    int* hist = reinterpret_cast<int*>(bin_smem + 3 * kBinTile);
    const int tid = threadIdx.x;
    const int base = blockIdx.x * kBinTile;
    load_event_tile(events, n, base, tile);
    int2 pl[kBinPer];
    int rank[kBinPer];
    if (use_smem) {
        for (int b = tid; b < nb1; b += kBinBlock) hist[b] = 0;
        __syncthreads();
#pragma unroll
        for (int q = 0; q < kBinPer; ++q) {
            const int i = base + q * kBinBlock + tid;
            pl[q] = i < n ? place[i] : make_int2(-1, 0);
            rank[q] = pl[q].x >= 0 ? atomicAdd(hist + pl[q].x, 1) : 0;
        }
        __syncthreads();
        for (int b = tid; b < nb1; b += kBinBlock) {
            const int c = hist[b];
            if (c) hist[b] = atomicAdd(cursors + b, c);       // count -> base of this block's run in bin b
        }
    }
    __syncthreads();
#pragma unroll
    for (int q = 0; q < kBinPer; ++q) {
        const int k = q * kBinBlock + tid, i = base + k;
        if (i >= n) continue;
        int pos;
        int2 pq;
        if (use_smem) { pq = pl[q]; pos = hist[pq.x] + rank[q]; }
        else { pq = place[i]; pos = atomicAdd(cursors + pq.x, 1); }
        const float zu = tile[3 * k], zd = tile[3 * k + 1], dl = tile[3 * k + 2];
        float4* dst = reinterpret_cast<float4*>(sorted + pos);
        if (pq.x == nb1 - 1) {
            dst[0] = make_float4(zu, zd, dl, 0.f);
        } else {
            const EventRec r = make_event_rec(zu, zd, dl, pq.y, p);
            dst[0] = make_float4(r.yoff, r.K2, r.B1, r.KB);
            dst[1] = make_float4(r.A0, r.A1, r.E0, r.E1);
            dst[2] = make_float4(r.D0, r.D1, r.D2, r.H2p);
            dst[3] = make_float4(r.Z0, r.T1, r.GS, __int_as_float(r.rows));
        }
    }
}

}  // namespace jpet
