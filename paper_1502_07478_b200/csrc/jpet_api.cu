// jpet_api.cu - C-ABI of include/jpet.h: argument checks, workspace, kernel launches.  No torch types.
#include "../../include/jpet.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>

#include "mlem_kernels.cuh"

namespace {

using jpet::DevParams;

thread_local std::string g_err;
std::atomic<uint64_t> g_launches{0};
float g_a3_coef = 2.0f;
int64_t g_opt_replicas = 0;      // 0 = automatic
int64_t g_opt_variant = -1;      // -1 = automatic
int64_t g_opt_ctas_per_sm = 0;   // 0 = automatic
constexpr int64_t kMaxBatch = 10000000;          // events per launch (BASELINE config 5: 10M-event batches)
constexpr int64_t kStageBytes = 4ll << 30;       // device staging budget of the host-buffer calls

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define CUDA_TRY(expr)                                                                              \
    do {                                                                                            \
        cudaError_t _e = (expr);                                                                    \
        if (_e != cudaSuccess)                                                                      \
            return fail(JPET_E_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
    } while (0)

struct Workspace {
    // problem the workspace is currently set up for
    jpet_geometry geom{0, 0};
    jpet_sigmas sig{0, 0};
    jpet_grid grid{0, 0, 0};
    float a3 = 0;
    bool s_valid = false;
    bool open = false;          // between begin and end
    int M = 0, n_rep = 0;
    DevParams dp{};
    int variant = 0;
    // device buffers
    float* s = nullptr;
    float* w = nullptr;
    float* acc = nullptr;
    float* rho_a = nullptr;
    float* rho_b = nullptr;
    unsigned long long* counters = nullptr;
    size_t cap_M = 0, cap_acc = 0;
    float* stage = nullptr;     // event staging for the host-buffer calls
    size_t cap_stage = 0;       // bytes
    cudaStream_t copy_stream = nullptr, compute_stream = nullptr;
    cudaEvent_t ev_copy[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr};
    int sm_count = 0;
    int device = -1;
} g_ws;

int validate(const jpet_geometry* g, const jpet_sigmas* sg, const jpet_grid* gr) {
    if (!g || !gr) return fail(JPET_E_INVAL, "NULL geometry or grid");
    if (!(g->R > 0.f) || !(g->L > 0.f) || !std::isfinite(g->R) || !std::isfinite(g->L))
        return fail(JPET_E_INVAL, "R and L must be positive and finite");
    if (gr->n_y <= 0 || gr->n_z <= 0 || !(gr->pixel > 0.f) || !std::isfinite(gr->pixel))
        return fail(JPET_E_INVAL, "n_y, n_z and pixel must be positive");
    if ((int64_t)gr->n_y * gr->n_z > (1ll << 28)) return fail(JPET_E_INVAL, "image too large");
    if (0.5 * (gr->n_y - 1) * (double)gr->pixel >= (double)g->R)
        return fail(JPET_E_INVAL, "grid reaches |y| >= R where Eq. 4 is singular");
    if (sg) {
        if (!(sg->sigma_z > 0.f) || !(sg->sigma_dl > 0.f) || !std::isfinite(sg->sigma_z) || !std::isfinite(sg->sigma_dl))
            return fail(JPET_E_INVAL, "sigmas must be positive and finite");
        // D = a.C^-1.a + 2 o.C^-1.b stays positive inside the 3-sigma ellipse when this ratio is < 1
        // (bound derived in DESIGN.md "Domain"); we ask for a factor 2 of margin.
        double ratio = (1.07 * sg->sigma_z + 1.8 * (double)sg->sigma_z * sg->sigma_z / sg->sigma_dl) / g->R;
        if (ratio > 0.5) return fail(JPET_E_INVAL, "sigmas too large against R: Eq. 7's square root could go non-positive");
        if (3.0 * sg->sigma_dl / gr->pixel > 60000.0 || 4.3 * sg->sigma_z / gr->pixel > 60000.0)
            return fail(JPET_E_INVAL, "ellipse spans too many pixels");
    }
    return JPET_OK;
}

int ensure_device() {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != g_ws.device) {
        if (g_ws.device >= 0) jpet_release();
        g_ws.device = dev;
        CUDA_TRY(cudaDeviceGetAttribute(&g_ws.sm_count, cudaDevAttrMultiProcessorCount, dev));
    }
    return JPET_OK;
}

int ensure_images(int M, int n_rep) {
    if ((size_t)M > g_ws.cap_M) {
        cudaFree(g_ws.s); cudaFree(g_ws.w); cudaFree(g_ws.rho_a); cudaFree(g_ws.rho_b);
        g_ws.s = g_ws.w = g_ws.rho_a = g_ws.rho_b = nullptr;
        g_ws.cap_M = 0;
        CUDA_TRY(cudaMalloc(&g_ws.s, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&g_ws.w, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&g_ws.rho_a, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&g_ws.rho_b, sizeof(float) * M));
        g_ws.cap_M = M;
        g_ws.s_valid = false;
    }
    if ((size_t)M * n_rep > g_ws.cap_acc) {
        cudaFree(g_ws.acc);
        g_ws.acc = nullptr;
        g_ws.cap_acc = 0;
        CUDA_TRY(cudaMalloc(&g_ws.acc, sizeof(float) * (size_t)M * n_rep));
        g_ws.cap_acc = (size_t)M * n_rep;
    }
    if (!g_ws.counters) CUDA_TRY(cudaMalloc(&g_ws.counters, 2 * sizeof(unsigned long long)));
    return JPET_OK;
}

// ---- event-kernel variants ------------------------------------------------------------------------------
struct Variant { int W, NW, NIT, threads; };
constexpr Variant kVariants[] = {
    {8, 1, 32, 256},    // 0: warp per event, 8-pixel segments, 128 cached segments
    {16, 1, 32, 256},   // 1: warp per event, 16-pixel segments, 64 cached segments
    {16, 4, 32, 256},   // 2: 4 warps per event, 16-pixel segments, 256 cached segments
    {16, 8, 24, 256},   // 3: 8 warps per event, 16-pixel segments, 384 cached segments
    {32, 4, 32, 256},   // 4: 4 warps per event, 32-pixel segments, 128 cached segments
    {8, 2, 32, 256},    // 5: 2 warps per event, 8-pixel segments, 256 cached segments
};
constexpr int kNumVariants = sizeof(kVariants) / sizeof(kVariants[0]);

template <int W, int NW, int NIT, int THREADS>
int launch_events(const float* events, int64_t n, const DevParams& dp, const float* w, float* acc, int M, int n_rep,
                  unsigned long long* counters, cudaStream_t stream) {
    auto kern = jpet::mlem_events_kernel<W, NW, NIT, THREADS>;
    constexpr int GROUPS = THREADS / (NW * 32);
    size_t rows_bytes = (size_t)dp.nrow_max * sizeof(jpet::RowRec);
    size_t seg_bytes = (((size_t)dp.nseg_max * 4 + 15) / 16) * 16;
    size_t group_bytes = rows_bytes + seg_bytes + 16 * ((NW * 4 + 15) / 16);
    size_t smem = group_bytes * GROUPS;
    if (smem > 220 * 1024) return fail(JPET_E_INVAL, "ellipse tables (%zu B) exceed shared memory; use a wider variant", smem);
    static size_t attr_set = 0;
    if (smem > 48 * 1024 && smem > attr_set) {
        CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = smem;
    }
    int per_sm = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, THREADS, smem));
    if (per_sm < 1) return fail(JPET_E_CUDA, "event kernel does not fit on an SM");
    if (g_opt_ctas_per_sm > 0) per_sm = (int)std::min<int64_t>(per_sm, g_opt_ctas_per_sm);
    int64_t want = (n + GROUPS - 1) / GROUPS;
    int grid = (int)std::min<int64_t>((int64_t)g_ws.sm_count * per_sm, std::max<int64_t>(want, 1));
    kern<<<grid, THREADS, smem, stream>>>(events, (long long)n, dp, w, acc, (long long)M, n_rep, counters);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

int dispatch_events(int variant, const float* events, int64_t n, const DevParams& dp, const float* w, float* acc, int M,
                    int n_rep, unsigned long long* counters, cudaStream_t stream) {
    switch (variant) {
        case 0: return launch_events<8, 1, 32, 256>(events, n, dp, w, acc, M, n_rep, counters, stream);
        case 1: return launch_events<16, 1, 32, 256>(events, n, dp, w, acc, M, n_rep, counters, stream);
        case 2: return launch_events<16, 4, 32, 256>(events, n, dp, w, acc, M, n_rep, counters, stream);
        case 3: return launch_events<16, 8, 24, 256>(events, n, dp, w, acc, M, n_rep, counters, stream);
        case 4: return launch_events<32, 4, 32, 256>(events, n, dp, w, acc, M, n_rep, counters, stream);
        case 5: return launch_events<8, 2, 32, 256>(events, n, dp, w, acc, M, n_rep, counters, stream);
        default: return fail(JPET_E_INVAL, "unknown kernel variant %d", variant);
    }
}

// Constants of the event kernel, computed in double and rounded once.
void make_params(const jpet_geometry& g, const jpet_sigmas& sg, const jpet_grid& gr, float a3, int W, DevParams* out) {
    DevParams p{};
    const double LH = 0.72134752044448170368;
    double iz2 = 1.0 / ((double)sg.sigma_z * sg.sigma_z), il2 = 1.0 / ((double)sg.sigma_dl * sg.sigma_dl);
    double px = gr.pixel;
    p.n_y = gr.n_y; p.n_z = gr.n_z;
    p.px = (float)px; p.inv_px = (float)(1.0 / px);
    p.y0 = (float)(-0.5 * (gr.n_y - 1) * px); p.z0 = (float)(-0.5 * (gr.n_z - 1) * px);
    p.inv2R = (float)(1.0 / (2.0 * g.R)); p.R2 = (float)((double)g.R * g.R);
    p.hy_coef = (float)(1.5 * sg.sigma_dl);
    p.half_sz2 = (float)(0.5 * (double)sg.sigma_z * sg.sigma_z);
    p.c1s = (float)(-LH * 2.0 * iz2);
    p.c2k = (float)(4.0 * il2);
    p.ak = (float)(-2.0 * iz2);
    p.bk = (float)(2.0 * a3 * il2);
    p.d1k = (float)(2.0 * iz2);
    p.d2k = (float)((double)a3 * a3 * il2);
    p.d3k = (float)(4.0 * il2);
    // capacities: rows <= 3 sigma_dl / px + 1; pixels <= area/px^2 + longest chord/px + rows (Riemann-sum bound)
    double rows = std::floor(3.0 * sg.sigma_dl / px) + 3.0;
    double chord = 2.0 * 3.0 * sg.sigma_z / std::sqrt(2.0) / px + 2.0;
    double area = 9.0 * M_PI * sg.sigma_z * sg.sigma_dl / (2.0 * std::sqrt(2.0)) / (px * px);
    rows = std::min(rows, (double)gr.n_y);
    double pix = area + chord + rows;
    p.nrow_max = (int)rows;
    p.nseg_max = (int)(pix / W + rows) + 8;
    *out = p;
}

int choose_variant(const jpet_sigmas& sg, const jpet_grid& gr) {
    if (g_opt_variant >= 0) return (int)g_opt_variant;
    double area = 9.0 * M_PI * sg.sigma_z * sg.sigma_dl / (2.0 * std::sqrt(2.0)) / ((double)gr.pixel * gr.pixel);
    if (area <= 900.0) return 0;
    if (area <= 3000.0) return 2;
    return 3;
}

int choose_replicas(int M) {
    if (g_opt_replicas > 0) return (int)g_opt_replicas;
    (void)M;
    return 8;
}

bool same_problem(const jpet_geometry& g, const jpet_grid& gr) {
    return g_ws.s_valid && g_ws.geom.R == g.R && g_ws.geom.L == g.L && g_ws.grid.n_y == gr.n_y &&
           g_ws.grid.n_z == gr.n_z && g_ws.grid.pixel == gr.pixel;
}

int grid_for(int M) { return (M + 255) / 256; }

int do_begin(const jpet_geometry* g, const jpet_sigmas* sg, const jpet_grid* gr, const float* rho_in, cudaStream_t st) {
    int rc = validate(g, sg, gr);
    if (rc) return rc;
    if (!sg) return fail(JPET_E_INVAL, "NULL sigmas");
    if (!rho_in) return fail(JPET_E_INVAL, "NULL rho_in");
    if ((rc = ensure_device())) return rc;
    const int M = gr->n_y * gr->n_z;
    const int n_rep = choose_replicas(M);
    if ((rc = ensure_images(M, n_rep))) return rc;
    if (!same_problem(*g, *gr)) {
        jpet::sensitivity_kernel<<<grid_for(M), 256, 0, st>>>(g_ws.s, gr->n_y, gr->n_z, gr->pixel, g->R, g->L);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
        g_ws.geom = *g; g_ws.grid = *gr; g_ws.s_valid = true;
    }
    g_ws.sig = *sg; g_ws.a3 = g_a3_coef; g_ws.M = M; g_ws.n_rep = n_rep;
    g_ws.variant = choose_variant(*sg, *gr);
    if (g_ws.variant < 0 || g_ws.variant >= kNumVariants) return fail(JPET_E_INVAL, "unknown kernel variant");
    make_params(*g, *sg, *gr, g_a3_coef, kVariants[g_ws.variant].W, &g_ws.dp);
    jpet::prepass_kernel<<<grid_for(M), 256, 0, st>>>(g_ws.s, rho_in, g_ws.w, g_ws.acc, M, n_rep, g_ws.counters);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    g_ws.open = true;
    return JPET_OK;
}

int do_accumulate(const float* events, int64_t n, cudaStream_t st) {
    if (!g_ws.open) return fail(JPET_E_INVAL, "jpet_mlem_accumulate without jpet_mlem_begin");
    if (n < 0) return fail(JPET_E_INVAL, "n < 0");
    if (n > 0 && !events) return fail(JPET_E_INVAL, "NULL events");
    for (int64_t off = 0; off < n; off += kMaxBatch) {
        int64_t nb = std::min(kMaxBatch, n - off);
        int rc = dispatch_events(g_ws.variant, events + 3 * off, nb, g_ws.dp, g_ws.w, g_ws.acc, g_ws.M, g_ws.n_rep,
                                 g_ws.counters, st);
        if (rc) return rc;
    }
    return JPET_OK;
}

int do_end(const float* rho_in, float* rho_out, cudaStream_t st) {
    if (!g_ws.open) return fail(JPET_E_INVAL, "jpet_mlem_end without jpet_mlem_begin");
    if (!rho_in || !rho_out) return fail(JPET_E_INVAL, "NULL image pointer");
    jpet::finalise_kernel<<<grid_for(g_ws.M), 256, 0, st>>>(g_ws.s, rho_in, g_ws.acc, rho_out, g_ws.M, g_ws.n_rep);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    g_ws.open = false;
    return JPET_OK;
}

int ensure_host_path(size_t stage_bytes) {
    if (!g_ws.copy_stream) {
        CUDA_TRY(cudaStreamCreateWithFlags(&g_ws.copy_stream, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&g_ws.compute_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CUDA_TRY(cudaEventCreateWithFlags(&g_ws.ev_copy[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&g_ws.ev_done[i], cudaEventDisableTiming));
        }
    }
    if (stage_bytes > g_ws.cap_stage) {
        cudaFree(g_ws.stage);
        g_ws.stage = nullptr;
        g_ws.cap_stage = 0;
        CUDA_TRY(cudaMalloc(&g_ws.stage, stage_bytes));
        g_ws.cap_stage = stage_bytes;
    }
    return JPET_OK;
}

// One iteration's accumulate phase from host events.  resident_in: events already in stage[0..n).
// If everything fits the staging buffer it is filled chunk by chunk (copy of chunk c+1 overlaps compute of chunk c)
// and left resident; otherwise two chunk-sized slots are used as a ring.
int accumulate_from_host(const float* events_host, int64_t n, int64_t chunk, bool fits, bool resident_in) {
    cudaStream_t cs = g_ws.copy_stream, ks = g_ws.compute_stream;
    if (resident_in) return do_accumulate(g_ws.stage, n, ks);
    int c = 0;
    for (int64_t off = 0; off < n; off += chunk, ++c) {
        int64_t nb = std::min(chunk, n - off);
        int slot = c & 1;
        float* dst = fits ? g_ws.stage + 3 * off : g_ws.stage + 3 * (int64_t)slot * chunk;
        if (!fits && c >= 2) CUDA_TRY(cudaStreamWaitEvent(cs, g_ws.ev_done[slot], 0));   // slot free again
        CUDA_TRY(cudaMemcpyAsync(dst, events_host + 3 * off, sizeof(float) * 3 * nb, cudaMemcpyHostToDevice, cs));
        CUDA_TRY(cudaEventRecord(g_ws.ev_copy[slot], cs));
        CUDA_TRY(cudaStreamWaitEvent(ks, g_ws.ev_copy[slot], 0));
        int rc = do_accumulate(dst, nb, ks);
        if (rc) return rc;
        if (!fits) CUDA_TRY(cudaEventRecord(g_ws.ev_done[slot], ks));
    }
    return JPET_OK;
}

int reconstruct_host_impl(const float* events_host, int64_t n, const jpet_geometry* g, const jpet_sigmas* sg,
                          const jpet_grid* gr, const float* rho_init_host, float* rho_out_host, int32_t n_iter,
                          int64_t chunk) {
    int rc = validate(g, sg, gr);
    if (rc) return rc;
    if (!sg) return fail(JPET_E_INVAL, "NULL sigmas");
    if (n < 0 || n_iter < 0) return fail(JPET_E_INVAL, "n < 0 or n_iter < 0");
    if ((n > 0 && !events_host) || !rho_out_host) return fail(JPET_E_INVAL, "NULL host pointer");
    if ((rc = ensure_device())) return rc;
    const int M = gr->n_y * gr->n_z;
    if ((rc = ensure_images(M, choose_replicas(M)))) return rc;
    if (chunk <= 0) chunk = 2000000;
    chunk = std::min<int64_t>(chunk, std::max<int64_t>(n, 1));
    const bool fits = (int64_t)sizeof(float) * 3 * n <= kStageBytes;
    size_t stage_bytes = fits ? sizeof(float) * 3 * (size_t)std::max<int64_t>(n, 1) : sizeof(float) * 3 * 2 * (size_t)chunk;
    if ((rc = ensure_host_path(stage_bytes))) return rc;
    cudaStream_t ks = g_ws.compute_stream;
    float* cur = g_ws.rho_a;
    float* nxt = g_ws.rho_b;
    if (rho_init_host) {
        CUDA_TRY(cudaMemcpyAsync(cur, rho_init_host, sizeof(float) * M, cudaMemcpyHostToDevice, ks));
    } else {
        jpet::ones_kernel<<<grid_for(M), 256, 0, ks>>>(cur, M);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
    }
    for (int it = 0; it < n_iter; ++it) {
        if ((rc = do_begin(g, sg, gr, cur, ks))) return rc;
        if ((rc = accumulate_from_host(events_host, n, chunk, fits, fits && it > 0))) return rc;
        if ((rc = do_end(cur, nxt, ks))) return rc;
        std::swap(cur, nxt);
    }
    CUDA_TRY(cudaMemcpyAsync(rho_out_host, cur, sizeof(float) * M, cudaMemcpyDeviceToHost, ks));
    CUDA_TRY(cudaStreamSynchronize(ks));
    CUDA_TRY(cudaStreamSynchronize(g_ws.copy_stream));
    return JPET_OK;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------
extern "C" {

int jpet_sensitivity(const jpet_geometry* geometry, const jpet_grid* grid, float* s_dev, void* cuda_stream) {
    g_err.clear();
    int rc = validate(geometry, nullptr, grid);
    if (rc) return rc;
    if (!s_dev) return fail(JPET_E_INVAL, "NULL s_dev");
    const int M = grid->n_y * grid->n_z;
    jpet::sensitivity_kernel<<<grid_for(M), 256, 0, (cudaStream_t)cuda_stream>>>(s_dev, grid->n_y, grid->n_z, grid->pixel,
                                                                               geometry->R, geometry->L);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

int jpet_mlem_begin(const jpet_geometry* geometry, const jpet_sigmas* sigmas, const jpet_grid* grid,
                    const float* rho_in_dev, void* cuda_stream) {
    g_err.clear();
    return do_begin(geometry, sigmas, grid, rho_in_dev, (cudaStream_t)cuda_stream);
}

int jpet_mlem_accumulate(const float* events_dev, int64_t n_batch, void* cuda_stream) {
    g_err.clear();
    return do_accumulate(events_dev, n_batch, (cudaStream_t)cuda_stream);
}

int jpet_mlem_end(const float* rho_in_dev, float* rho_out_dev, void* cuda_stream) {
    g_err.clear();
    return do_end(rho_in_dev, rho_out_dev, (cudaStream_t)cuda_stream);
}

int jpet_mlem_iterate(const float* events_dev, int64_t n, const jpet_geometry* geometry, const jpet_sigmas* sigmas,
                      const jpet_grid* grid, const float* rho_in_dev, float* rho_out_dev, void* cuda_stream) {
    g_err.clear();
    int rc = validate(geometry, sigmas, grid);
    if (rc) return rc;
    if (n < 0) return fail(JPET_E_INVAL, "n < 0");
    if (n > 0 && !events_dev) return fail(JPET_E_INVAL, "NULL events");
    if (!rho_in_dev || !rho_out_dev) return fail(JPET_E_INVAL, "NULL image pointer");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = do_begin(geometry, sigmas, grid, rho_in_dev, st))) return rc;
    if ((rc = do_accumulate(events_dev, n, st))) { g_ws.open = false; return rc; }
    return do_end(rho_in_dev, rho_out_dev, st);
}

int jpet_reconstruct(const float* events_dev, int64_t n, const jpet_geometry* geometry, const jpet_sigmas* sigmas,
                     const jpet_grid* grid, const float* rho_init_dev, float* rho_out_dev, int32_t n_iter,
                     void* cuda_stream) {
    g_err.clear();
    int rc = validate(geometry, sigmas, grid);
    if (rc) return rc;
    if (!sigmas) return fail(JPET_E_INVAL, "NULL sigmas");
    if (n < 0 || n_iter < 0) return fail(JPET_E_INVAL, "n < 0 or n_iter < 0");
    if ((n > 0 && !events_dev) || !rho_out_dev) return fail(JPET_E_INVAL, "NULL pointer");
    if ((rc = ensure_device())) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int M = grid->n_y * grid->n_z;
    if ((rc = ensure_images(M, choose_replicas(M)))) return rc;
    // ping-pong through the workspace so that rho_out may alias rho_init and is written once per iteration
    const float* cur = rho_init_dev;
    if (!cur) {
        jpet::ones_kernel<<<grid_for(M), 256, 0, st>>>(g_ws.rho_a, M);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
        cur = g_ws.rho_a;
    }
    if (n_iter == 0) {
        if (cur != rho_out_dev) CUDA_TRY(cudaMemcpyAsync(rho_out_dev, cur, sizeof(float) * M, cudaMemcpyDeviceToDevice, st));
        return JPET_OK;
    }
    for (int it = 0; it < n_iter; ++it) {
        float* nxt = (it == n_iter - 1) ? rho_out_dev : (cur == g_ws.rho_a ? g_ws.rho_b : g_ws.rho_a);
        if ((rc = do_begin(geometry, sigmas, grid, cur, st))) return rc;
        if ((rc = do_accumulate(events_dev, n, st))) { g_ws.open = false; return rc; }
        if ((rc = do_end(cur, nxt, st))) return rc;
        cur = nxt;
    }
    return JPET_OK;
}

int jpet_mlem_iterate_host(const float* events_host, int64_t n, const jpet_geometry* geometry, const jpet_sigmas* sigmas,
                           const jpet_grid* grid, const float* rho_in_host, float* rho_out_host, int64_t chunk_events) {
    g_err.clear();
    if (!rho_in_host) return fail(JPET_E_INVAL, "NULL rho_in_host");
    return reconstruct_host_impl(events_host, n, geometry, sigmas, grid, rho_in_host, rho_out_host, 1, chunk_events);
}

int jpet_reconstruct_host(const float* events_host, int64_t n, const jpet_geometry* geometry, const jpet_sigmas* sigmas,
                          const jpet_grid* grid, const float* rho_init_host, float* rho_out_host, int32_t n_iter,
                          int64_t chunk_events) {
    g_err.clear();
    return reconstruct_host_impl(events_host, n, geometry, sigmas, grid, rho_init_host, rho_out_host, n_iter, chunk_events);
}

int jpet_get_counters(uint64_t* n_evals_host, uint64_t* n_skipped_host, void* cuda_stream) {
    g_err.clear();
    if (!g_ws.counters) return fail(JPET_E_INVAL, "no iteration has been run");
    unsigned long long h[2];
    CUDA_TRY(cudaMemcpyAsync(h, g_ws.counters, sizeof h, cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
    CUDA_TRY(cudaStreamSynchronize((cudaStream_t)cuda_stream));
    if (n_evals_host) *n_evals_host = h[0];
    if (n_skipped_host) *n_skipped_host = h[1];
    return JPET_OK;
}

int jpet_count_evals(const float* events_dev, int64_t n, const jpet_geometry* geometry, const jpet_sigmas* sigmas,
                     const jpet_grid* grid, uint64_t* n_evals_host, uint64_t* n_skipped_host, void* cuda_stream) {
    g_err.clear();
    int rc = validate(geometry, sigmas, grid);
    if (rc) return rc;
    if (!sigmas) return fail(JPET_E_INVAL, "NULL sigmas");
    if (n < 0 || (n > 0 && !events_dev)) return fail(JPET_E_INVAL, "bad events");
    if ((rc = ensure_device())) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned long long* d = nullptr;
    CUDA_TRY(cudaMalloc(&d, 2 * sizeof(unsigned long long)));
    CUDA_TRY(cudaMemsetAsync(d, 0, 2 * sizeof(unsigned long long), st));
    DevParams dp;
    make_params(*geometry, *sigmas, *grid, g_a3_coef, 8, &dp);
    dp.nrow_max = grid->n_y;
    if (n > 0) {
        int blocks = (int)std::min<int64_t>((n + 255) / 256, (int64_t)g_ws.sm_count * 8);
        jpet::count_evals_kernel<<<blocks, 256, 0, st>>>(events_dev, (long long)n, dp, d);
        g_launches++;
    }
    unsigned long long h[2] = {0, 0};
    cudaError_t e = cudaMemcpyAsync(h, d, sizeof h, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d);
    if (e != cudaSuccess) return fail(JPET_E_CUDA, "count_evals: %s", cudaGetErrorString(e));
    if (n_evals_host) *n_evals_host = h[0];
    if (n_skipped_host) *n_skipped_host = h[1];
    return JPET_OK;
}

int jpet_set_a3_coef(float k) {
    g_err.clear();
    if (!std::isfinite(k)) return fail(JPET_E_INVAL, "a3 coefficient must be finite");
    g_a3_coef = k;
    return JPET_OK;
}

float jpet_get_a3_coef(void) { return g_a3_coef; }

int jpet_set_option(const char* name, int64_t value) {
    g_err.clear();
    if (!name) return fail(JPET_E_INVAL, "NULL option name");
    if (!strcmp(name, "replicas")) {
        if (value < 0 || value > 64) return fail(JPET_E_INVAL, "replicas must be 0 (auto) .. 64");
        g_opt_replicas = value;
    } else if (!strcmp(name, "variant")) {
        if (value < -1 || value >= kNumVariants) return fail(JPET_E_INVAL, "variant must be -1 (auto) .. %d", kNumVariants - 1);
        g_opt_variant = value;
    } else if (!strcmp(name, "ctas_per_sm")) {
        if (value < 0 || value > 32) return fail(JPET_E_INVAL, "ctas_per_sm must be 0 (auto) .. 32");
        g_opt_ctas_per_sm = value;
    } else {
        return fail(JPET_E_INVAL, "unknown option '%s'", name);
    }
    return JPET_OK;
}

int64_t jpet_get_option(const char* name) {
    if (!name) return -1;
    if (!strcmp(name, "replicas")) return g_opt_replicas;
    if (!strcmp(name, "variant")) return g_opt_variant;
    if (!strcmp(name, "ctas_per_sm")) return g_opt_ctas_per_sm;
    if (!strcmp(name, "last_variant")) return g_ws.variant;
    if (!strcmp(name, "last_replicas")) return g_ws.n_rep;
    return -1;
}

uint64_t jpet_launch_count(void) { return g_launches.load(); }

void jpet_release(void) {
    cudaFree(g_ws.s); cudaFree(g_ws.w); cudaFree(g_ws.acc); cudaFree(g_ws.rho_a); cudaFree(g_ws.rho_b);
    cudaFree(g_ws.counters); cudaFree(g_ws.stage);
    for (int i = 0; i < 2; ++i) {
        if (g_ws.ev_copy[i]) cudaEventDestroy(g_ws.ev_copy[i]);
        if (g_ws.ev_done[i]) cudaEventDestroy(g_ws.ev_done[i]);
    }
    if (g_ws.copy_stream) cudaStreamDestroy(g_ws.copy_stream);
    if (g_ws.compute_stream) cudaStreamDestroy(g_ws.compute_stream);
    int dev = g_ws.device, sms = g_ws.sm_count;
    g_ws = Workspace{};
    g_ws.device = dev;
    g_ws.sm_count = sms;
}

const char* jpet_last_error(void) { return g_err.c_str(); }

int jpet_abi_version(void) { return JPET_ABI_VERSION; }

}  // extern "C"
