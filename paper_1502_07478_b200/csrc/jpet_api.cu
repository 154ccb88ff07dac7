// jpet_api.cu - C-ABI of include/jpet.h: argument checks, per-device workspaces, the plan, kernel launches.
// No torch types.  The tiled event kernel is instantiated in rows_inst_*.cu (one file per group of shapes, compiled in
// parallel by build.py) and reached through launch_rows_shape() of rows_launch.h.
#include "../../include/jpet.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <memory>
#include <string>
#include <vector>

#include "generator.cuh"
#include "histogram.cuh"
#include "image_kernels.cuh"
#include "mlem_direct.cuh"
#include "rows_launch.h"
#include "sort_kernels.cuh"
#include "task_table.h"

namespace jpet_host {
std::atomic<uint64_t> g_launches{0};
thread_local std::string g_err;

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}
}  // namespace jpet_host

namespace jpet_host {
int launch_rows_shape(const RowsLaunch& rl) {
    int rc = launch_rows_group0(rl);
    if (rc == -100) rc = launch_rows_group1(rl);
    if (rc == -100) rc = launch_rows_group2(rl);
    if (rc == -100) rc = launch_rows_group3(rl);
    if (rc == -100) rc = fail(JPET_E_INVAL, "unknown kernel shape %d", rl.shape);
    return rc;
}
}  // namespace jpet_host

namespace {

using jpet::DevParams;
using jpet_host::BinSet;
using jpet_host::fail;
using jpet_host::g_err;
using jpet_host::g_launches;
using jpet_host::kNumShapes;
using jpet_host::kShapes;
using jpet_host::Shape;

// ---- process-wide settings (include/jpet.h: a3 coefficient, gamma, sigma_z edge coefficient, tuning options) ------
struct Options {
    float a3_coef = 2.0f;
    float gamma = 0.0f;           // off-diagonal coefficient of C^-1 (Eq. 12); 0 = the paper's diagonal case
    float sz_eta = 0.0f;          // sigma_z(z) = sigma_z (1 + eta (2z/L)^2); 0 = constant
    int64_t force_direct = 0;     // 1 = every event takes the direct (global-memory) path
    int64_t chunk = 0;            // events per work item, 0 = automatic
    int64_t sz = 0;               // sub-tile width in pixels, 0 = automatic
    int64_t time_kernel = 0;      // 1 = bracket the tiled event kernel with CUDA events (bench.py's roofline)
    int64_t variant = -1;         // shape id, -1 = automatic
    int64_t pdl = 1;              // 1 = launch the kernels of an iteration with programmatic stream serialisation
    int64_t poly_off = 0;         // 1 = never pick a polynomial-exponent shape automatically
    int64_t cls_off = 0;          // 1 = no per-event degree classes
    int64_t ctas_per_sm = 0;      // 0 = automatic
    int64_t stage_bytes = 0;      // device staging budget of the host-buffer calls; 0 = default
    int64_t exact_kernel = 0;     // > 0: theta-quadrature nodes of the exact-kernel mode
} g_opt;
constexpr int64_t kMaxBatch = 10000000;          // events per launch (BASELINE config 5: 10M-event batches)
constexpr int64_t kStageDefault = 4ll << 30;

#define CUDA_TRY(expr)                                                                              \
    do {                                                                                            \
        cudaError_t _e = (expr);                                                                    \
        if (_e != cudaSuccess) {                                                                    \
            (void)cudaGetLastError(); /* reported here: do not leave it for an unrelated later call */ \
            return fail(JPET_E_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
        }                                                                                           \
    } while (0)

// Everything the plan depends on; compared field by field (no padding bytes involved).
struct PlanKey {
    jpet_geometry g{0, 0};
    jpet_sigmas sg{0, 0};
    jpet_grid gr{0, 0, 0};
    float a3 = 0, gamma = 0, sz_eta = 0;
    int64_t variant = 0, sz = 0, chunk = 0, force_direct = 0, poly_off = 0, exact = 0, cls_off = 0;
    bool operator==(const PlanKey& o) const {
        return g.R == o.g.R && g.L == o.g.L && sg.sigma_z == o.sg.sigma_z && sg.sigma_dl == o.sg.sigma_dl && gr.n_y == o.gr.n_y &&
               gr.n_z == o.gr.n_z && gr.pixel == o.gr.pixel && a3 == o.a3 && gamma == o.gamma && sz_eta == o.sz_eta &&
               variant == o.variant && sz == o.sz && chunk == o.chunk && force_direct == o.force_direct && poly_off == o.poly_off &&
               exact == o.exact && cls_off == o.cls_off;
    }
};

// One per CUDA device (the current device of the calling thread selects it).
struct Workspace {
    int device = -1;
    int sm_count = 0;
    // problem the workspace is currently set up for
    jpet_geometry geom{0, 0};
    jpet_sigmas sig{0, 0};
    jpet_grid grid{0, 0, 0};
    bool s_valid = false;
    bool open = false;          // between begin and end
    int M = 0;
    jpet_host::RowsPlan plan;   // DevParams, shape, shared memory, task table pointer
    PlanKey plan_key;
    bool plan_valid = false;
    // device buffers
    float* s = nullptr;
    float* wT = nullptr;
    float* accT = nullptr;
    float* rho_a = nullptr;
    float* rho_b = nullptr;
    unsigned long long* counters = nullptr;      // 0 evals, 1 skipped, 2 overflow flags, 3 scratch
    size_t cap_M = 0;
    int2* place = nullptr;      // scratch of the binning pass: (bin, packed rows) per event
    size_t cap_place = 0;
    int* counts = nullptr;      // [nb + 1] counts, then [nb + 1] cursors
    size_t cap_counts = 0;
    int counts_clean_nb = -1;   // bin count of the layout the (zeroed) counts buffer was last used with
    BinSet scratch;             // used by iterate / accumulate
    std::vector<BinSet> kept;   // used by reconstruct: one per batch, binned once
    float* kept_sorted = nullptr;
    size_t cap_kept_sorted = 0;
    float* stage = nullptr;     // event staging for the host-buffer calls
    size_t cap_stage = 0;       // bytes
    cudaStream_t copy_stream = nullptr, compute_stream = nullptr;
    cudaEvent_t ev_copy[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr};
    bool slot_used[2] = {false, false};          // ring slots of the staging buffer that a kernel may still be reading
    uint32_t* tab = nullptr;    // task table (device copy of tab_host)
    size_t cap_tab = 0;
    std::vector<uint32_t> tab_host, tab_uploaded;
    bool sort_attr_set = false;
    // ordering between streams: every call waits, on its stream, for the previous call's work
    cudaEvent_t ev_last = nullptr;
    cudaStream_t last_stream = nullptr;
    bool have_last = false;
    // CUDA-event pairs around the tiled event kernel launches since the last begin ("time_kernel")
    std::vector<cudaEvent_t> tk;
    size_t tk_used = 0;
};
std::map<int, std::unique_ptr<Workspace>> g_ctx;
int g_last_device = -1;      // device of the most recent call that touched a workspace (jpet_get_option "last_*")

int current_ws(Workspace** out) {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    auto& slot = g_ctx[dev];
    if (!slot) {
        slot.reset(new Workspace());
        slot->device = dev;
        CUDA_TRY(cudaDeviceGetAttribute(&slot->sm_count, cudaDevAttrMultiProcessorCount, dev));
    }
    g_last_device = dev;
    *out = slot.get();
    return JPET_OK;
}

// The workspace of the calling thread's current device if one exists (accumulate / end / counters follow a begin).
Workspace* device_ws() {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return nullptr;
    auto it = g_ctx.find(dev);
    if (it == g_ctx.end()) return nullptr;
    g_last_device = dev;
    return it->second.get();
}

Workspace* last_ws() {
    auto it = g_ctx.find(g_last_device);
    return it == g_ctx.end() ? nullptr : it->second.get();
}

// Stream ordering (include/jpet.h): the workspace is used by one stream at a time.
int enter(Workspace& w, cudaStream_t st) {
    if (w.have_last && w.last_stream != st) CUDA_TRY(cudaStreamWaitEvent(st, w.ev_last, 0));
    return JPET_OK;
}
int leave(Workspace& w, cudaStream_t st) {
    if (!w.ev_last) CUDA_TRY(cudaEventCreateWithFlags(&w.ev_last, cudaEventDisableTiming));
    CUDA_TRY(cudaEventRecord(w.ev_last, st));
    w.last_stream = st;
    w.have_last = true;
    return JPET_OK;
}

// Every way out of a call that has passed enter() - success or error - records the ordering event (the next call, on
// whatever stream, is ordered behind everything this call managed to queue), and a host-buffer call also waits for its
// two internal streams: no asynchronous copy may still be reading the caller's host buffers, and no ring slot may still
// be in flight, once the call has returned - also when it returns an error.  finish() is the success path and reports
// its own failures; the destructor covers the early returns and keeps the error text of the failure that caused them.
struct CallScope {
    Workspace& w;
    cudaStream_t st;
    bool host;
    bool done = false;
    CallScope(Workspace& w_, cudaStream_t st_, bool host_ = false) : w(w_), st(st_), host(host_) {}
    CallScope(const CallScope&) = delete;
    CallScope& operator=(const CallScope&) = delete;
    int finish() {
        done = true;
        int rc = leave(w, st);
        if (host) {
            cudaError_t e1 = cudaStreamSynchronize(st), e2 = cudaStreamSynchronize(w.copy_stream);
            if (!rc && (e1 != cudaSuccess || e2 != cudaSuccess)) {
                (void)cudaGetLastError();
                rc = fail(JPET_E_CUDA, "cudaStreamSynchronize failed: %s", cudaGetErrorString(e1 != cudaSuccess ? e1 : e2));
            }
        }
        return rc;
    }
    ~CallScope() {
        if (done) return;
        const std::string text = g_err;
        (void)leave(w, st);
        if (host) {
            (void)cudaStreamSynchronize(st);
            if (w.copy_stream) (void)cudaStreamSynchronize(w.copy_stream);
        }
        (void)cudaGetLastError();
        g_err = text;
    }
};

double sigma_z_max(const jpet_sigmas& sg) { return (double)sg.sigma_z * (1.0 + (double)g_opt.sz_eta); }

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
        // (bound derived in DESIGN.md "Domain"); we ask for a factor 2 of margin.  With a position-dependent sigma_z
        // the largest value (strip edge) enters.
        const double szm = sigma_z_max(*sg);
        double ratio = (1.07 * szm + 1.8 * szm * szm / sg->sigma_dl) / g->R;
        if (ratio > 0.5) return fail(JPET_E_INVAL, "sigmas too large against R: Eq. 7's square root could go non-positive");
        // Eq. 12 is positive definite for gamma^2 < 1 / (2 sigma_z^2 sigma_dl^2); half of that keeps D > 0 as well
        // (a.C^-1.a changes by at most 2 |gamma| k y sigma_z^2 sin(theta) / R of itself)
        if (std::fabs((double)g_opt.gamma) * std::sqrt(2.0) * szm * sg->sigma_dl > 0.5)
            return fail(JPET_E_INVAL, "|gamma| must be at most 0.5 / (sqrt(2) sigma_z sigma_dl) (Eq. 12 positive definite, D > 0)");
        if (3.0 * sg->sigma_dl / gr->pixel > 60000.0 || 4.3 * szm / gr->pixel > 60000.0)
            return fail(JPET_E_INVAL, "ellipse spans too many pixels");
    }
    return JPET_OK;
}

int ensure_images(Workspace& w, int M) {
    if ((size_t)M > w.cap_M) {
        cudaFree(w.s); cudaFree(w.wT); cudaFree(w.accT); cudaFree(w.rho_a); cudaFree(w.rho_b);
        w.s = w.wT = w.accT = w.rho_a = w.rho_b = nullptr;
        w.cap_M = 0;
        CUDA_TRY(cudaMalloc(&w.s, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&w.wT, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&w.accT, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&w.rho_a, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&w.rho_b, sizeof(float) * M));
        w.cap_M = M;
        w.s_valid = false;
    }
    if (!w.counters) CUDA_TRY(cudaMalloc(&w.counters, 4 * sizeof(unsigned long long)));
    return JPET_OK;
}

// Kernel launch with the programmatic-stream-serialisation attribute (PDL): the kernel may be scheduled while the
// previous kernel of the stream drains; every kernel launched this way starts with pdl_wait() (common.cuh), so it
// reads nothing the previous kernel wrote before that kernel has completed.  Hides most of the launch gaps between
// the eight kernels of an iteration (config 2: a 0.8 ms step).
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = g_opt.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// Events per work item for a batch of n events: the plan's size, halved (not below 64) while the batch would give fewer
// than three items per resident CTA (MINB CTAs per SM for the shape) - small batches are launch- and tail-bound
// (config 2, 10^6 events on 592 CTAs: 0.683 ms with 512 events per item, 0.716 ms with 1024).
int batch_chunk(const Workspace& w, int64_t n) {
    int chunk = w.plan.dp.chunk;
    if (g_opt.chunk > 0) return chunk;
    const int64_t ctas = (int64_t)w.sm_count * std::max(1, kShapes[std::min(std::max(w.plan.shape, 0), kNumShapes - 1)].MINB);
    while (chunk > 64 && n / chunk < 3 * ctas) chunk /= 2;
    return chunk;
}

// The tiled event kernel over the regular bins of a sorted batch, then the direct kernel over its last bin (all events
// when no region fits shared memory, or in the exact-kernel mode).
int run_binset(Workspace& w, BinSet& bs, cudaStream_t st) {
    const DevParams& dp = w.plan.dp;
    if (dp.t_max >= 0.f) {
        if (g_opt.time_kernel) {
            if (w.tk_used + 2 > w.tk.size()) {
                w.tk.resize(w.tk_used + 2, nullptr);
                CUDA_TRY(cudaEventCreate(&w.tk[w.tk_used])); CUDA_TRY(cudaEventCreate(&w.tk[w.tk_used + 1]));
            }
            CUDA_TRY(cudaEventRecord(w.tk[w.tk_used], st));
        }
        jpet_host::RowsLaunch rl;
        rl.bs = &bs; rl.plan = &w.plan; rl.wT = w.wT; rl.accT = w.accT; rl.tab = w.tab; rl.counters = w.counters;
        rl.sm_count = w.sm_count; rl.device = w.device; rl.stream = st; rl.pdl = g_opt.pdl != 0;
        rl.ctas_per_sm = (int)g_opt.ctas_per_sm;
        rl.max_items = bs.n / batch_chunk(w, bs.n) + (int64_t)dp.nby * dp.nbz * dp.n_cls + 1;
        rl.shape = w.plan.shape; rl.cls = 0;
        int rc = jpet_host::launch_rows_shape(rl);
        if (rc) return rc;
        if (dp.n_cls == 2) {                 // the events of degree class 1 on the degree-3 instance of the shape
            rl.shape = w.plan.shape_lo; rl.cls = 1;
            if ((rc = jpet_host::launch_rows_shape(rl))) return rc;
        }
        if (g_opt.time_kernel) { CUDA_TRY(cudaEventRecord(w.tk[w.tk_used + 1], st)); w.tk_used += 2; }
    }
    // the work counters are zero before the tiled kernels: bin_scan_kernel zeroes them and the direct kernel, the last
    // kernel of every run over a sorted set, zeroes them again (jpet_reconstruct sorts once and iterates)
    const int dgrid = dp.t_max >= 0.f ? w.sm_count : w.sm_count * 16;
    if (g_opt.exact_kernel > 0)
        CUDA_TRY(launch_pdl(jpet::mlem_rows_direct_kernel<true>, dim3(dgrid), dim3(128), 0, st, (const float*)bs.sorted, 16, bs.meta, dp,
                            (const float*)w.wT, w.accT, w.counters, (int)g_opt.exact_kernel));
    else
        CUDA_TRY(launch_pdl(jpet::mlem_rows_direct_kernel<false>, dim3(dgrid), dim3(128), 0, st, (const float*)bs.sorted, 16, bs.meta, dp,
                            (const float*)w.wT, w.accT, w.counters, 0));
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

// Constants of the event kernel (computed in double, rounded once), the tiling of the image into
// sub-tiles + halo regions, and the kernel shape.
void make_plan(const jpet_geometry& g, const jpet_sigmas& sg, const jpet_grid& gr, jpet_host::RowsPlan* out,
               std::vector<uint32_t>* tab_out = nullptr) {
    DevParams p{};
    const float a3 = g_opt.a3_coef, gamma = g_opt.gamma;
    const double LH = 0.72134752044448170368;
    const double eta = g_opt.sz_eta, szm = sigma_z_max(sg);          // largest sigma_z an event can see
    double iz2 = 1.0 / ((double)sg.sigma_z * sg.sigma_z), il2 = 1.0 / ((double)sg.sigma_dl * sg.sigma_dl);
    double px = gr.pixel;
    p.n_y = gr.n_y; p.n_z = gr.n_z;
    p.px = (float)px; p.inv_px = (float)(1.0 / px);
    p.y0 = (float)(-0.5 * (gr.n_y - 1) * px); p.z0 = (float)(-0.5 * (gr.n_z - 1) * px);
    p.inv2R = (float)(1.0 / (2.0 * g.R)); p.R2 = (float)((double)g.R * g.R); p.R = g.R;
    p.hy_coef = (float)(1.5 * sg.sigma_dl);
    p.half_sz2 = (float)(0.5 * (double)sg.sigma_z * sg.sigma_z);
    p.c1s = (float)(-LH * 2.0 * iz2);
    p.sq = (float)std::sqrt(LH * 2.0 * iz2);
    p.inv_sq = (float)(1.0 / std::sqrt(LH * 2.0 * iz2));
    p.pxs = (float)(px * std::sqrt(LH * 2.0 * iz2));
    p.H0p = (float)(9.0 * 0.5 * (double)sg.sigma_z * sg.sigma_z / (px * px));
    p.c2k = (float)(4.0 * il2);
    p.ak = (float)(-2.0 * iz2);
    p.bk = (float)(2.0 * a3 * il2);
    p.d1k = (float)(2.0 * iz2);
    p.d2k = (float)((double)a3 * a3 * il2);
    p.d3k = (float)(4.0 * il2);
    p.gB = (float)(4.0 * (double)gamma * g.R);
    p.gD0 = (float)(4.0 * (double)gamma * g.R * a3);
    p.sz_eta = (float)eta;
    p.inv_hL2 = (float)(4.0 / ((double)g.L * g.L));
    // ellipse extents in pixels: half height 1.5 sigma_dl cos(theta), half width 3 sqrt(sz^2/2 + sdl^2 sin^2/4) (App. B)
    double t_max = ((double)g.L + 8.0 * szm) / (2.0 * g.R);
    double sin2 = t_max * t_max / (1.0 + t_max * t_max);
    double hy = 1.5 * sg.sigma_dl / px;
    double hz = 3.0 * std::sqrt(0.5 * szm * szm + 0.25 * (double)sg.sigma_dl * sg.sigma_dl * sin2) / px;
    const double H0p_max = 9.0 * 0.5 * szm * szm / (px * px);       // half chord^2 at the centre row, widest event
    p.Hy = (int)std::ceil(hy) + 1;
    p.Hz = (int)std::ceil(hz) + 1;
    p.t_max = (float)t_max;
    // ellipse row counts a regular event can have (unclipped): hy_px * cos(theta) for |tan theta| <= t_max, +- rounding
    const int nr_hi = std::min(255, (int)std::floor(2.0 * hy) + 2);
    const int nr_lo = std::max(1, (int)std::floor(2.0 * hy / std::sqrt(1.0 + t_max * t_max)) - 1);
    std::vector<uint32_t> tab;
    auto fits = [&](const Shape& c) {
        return 2 * p.Hy + 4 <= c.HS && jpet_host::build_task_table(nr_lo, nr_hi, H0p_max, c.NWE, c.NJA, c.NJB, &tab);
    };
    int v = -1;
    if (g_opt.variant >= 0) v = (int)g_opt.variant;
    else {
        // degree of the exponent polynomial from the truncation bound (mlem_rows.cuh, poly_coeffs2):
        // |x| = |eps u / delta| <= xb, ba^2 / D <= eb inside the ellipse and the image.  A position-dependent sigma_z
        // adds the term Dl R to S y in alpha and eps (common.cuh): |Dl| / S <= dls, i.e. y grows by at most dls R.
        const double dls = ((1.0 + eta) * (1.0 + eta) - 1.0) / ((1.0 + eta) * (1.0 + eta) + 1.0);
        const double y_max = 0.5 * gr.n_y * px + dls * g.R, u_max = 3.0 * szm / std::sqrt(2.0), R2 = (double)g.R * g.R;
        // gamma (Eq. 12): delta changes by at most g_rel of itself, |b.C^-1.a| / sqrt(D) grows by at most g_ba
        const double ag = std::fabs((double)gamma);
        const double g_rel = 2.0 * ag * std::fabs((double)a3) * y_max * szm * szm * (t_max / std::sqrt(1.0 + t_max * t_max)) / g.R;
        const double g_ba = 6.0 / std::sqrt(2.0) * ag * szm * sg.sigma_dl;
        // |t| / sec^2 = |t| / (1 + t^2) grows up to |t| = 1, where it is 1/2, and falls beyond: its largest value over
        // |t| <= t_max is at t_max only while t_max < 1 (strips longer than 2 R reach |t| = 1)
        const double tf = t_max < 1.0 ? t_max / (1.0 + t_max * t_max) : 0.5;
        const double xb = 2.0 * tf * y_max * u_max / (R2 + y_max * y_max) / (0.95 - g_rel - 2.0 * dls * y_max * g.R / (R2 + y_max * y_max));
        const double eb = 1.1 * std::pow(3.0 * y_max / std::sqrt(R2 + y_max * y_max) + g_ba, 2.0);
        // What has to be small is the error of a kernel value against the event's largest one (the image tolerance is
        // relative to the image maximum).  At the fraction s = |u| / u_max of the central half chord |x| <= xb s; the tail
        // of ba^2 / D is e_2 v^2 |x|^(deg-1) / (1 - |x|) with e_2 v^2 = (alpha v - x beta)^2 / delta <= eb s^2 (1 + xb)^2, the
        // tail of ln D is |x|^(deg+1) / (deg + 1): both scale with s^(deg+1).  The kernel value there is at most
        // exp(-q (1 - eb/9) / 2) of the peak (b.C^-1.a is linear in b, so ba^2 / D <= (eb / 9) q, and q = b.C^-1.b >= 9 s^2),
        // times <= 1.05 for the D^-1/2 factor.  max over s in [0, 1] of s^n exp(-g s^2) is (n / (2 g e))^(n/2) when n <= 2 g,
        // else exp(-g).  low_degree_ok (common.cuh) is the same bound for one event.
        const double gw = 4.5 * std::max(0.0, 1.0 - eb / 9.0);
        auto wmax = [&](int n) { return 1.05 * (n < 2.0 * gw ? std::pow(n / (2.0 * gw * std::exp(1.0)), 0.5 * n) : std::exp(-gw)); };
        auto trunc_err = [&](int deg) {      // log2 units, weighted by the kernel value relative to the event's peak
            return 1.4427 * wmax(deg + 1) * (0.5 * eb * (1.0 + xb) * (1.0 + xb) * std::pow(xb, deg - 1) / (1.0 - xb) + 0.5 * std::pow(xb, deg + 1) / (deg + 1));
        };
        // among the degrees that meet the bound (a higher degree is only more accurate): the first shape of each degree
        // that holds the workload's ellipses (the list is ordered by size within a degree), then the one with the fewest
        // pixel slots per event, the lowest degree on a tie; no polynomial degree: the closed form
        const bool poly_ok = !g_opt.poly_off && xb > 0.0 && xb < 0.5;
        int best_slots = 0;
        for (int deg = 3; deg <= 5 && poly_ok; ++deg) {
            if (!(trunc_err(deg) <= 2e-5)) continue;
            for (int s = 0; s < kNumShapes; ++s) {
                if (kShapes[s].DEG != deg || !fits(kShapes[s])) continue;
                const int slots = 32 * kShapes[s].NWE * (kShapes[s].NJA + kShapes[s].NJB);
                if (v < 0 || slots < best_slots) { v = s; best_slots = slots; }
                break;
            }
        }
        for (int s = 0; s < kNumShapes && v < 0; ++s)
            if (kShapes[s].DEG == 0 && fits(kShapes[s])) v = s;
    }
    // no shape fits (or a forced shape does not): every event takes the direct path
    bool tiles_ok = v >= 0 && fits(kShapes[v]);
    if (v < 0) v = 0;
    // Degree classes: the bound above holds for the worst event the image can hold (largest |y|, largest tilt); most
    // events are far from it.  When the plan's degree is 4 or 5 and the shape has a degree-3 instance, the sort tests
    // every event against its OWN bound (low_degree_ok, common.cuh; gamma = 0 and constant sigma_z only) and the events
    // that pass are walked by the degree-3 instance (configs 2 and 4: 100 % / 77 % of the events, -6 % / -5 % time).
    int v_lo = -1;
    if (g_opt.variant < 0 && !g_opt.cls_off && tiles_ok && kShapes[v].DEG > 3 && kShapes[v].CLS && gamma == 0.f && eta == 0.0)
        for (int s = 0; s < kNumShapes && v_lo < 0; ++s)
            if (kShapes[s].DEG == 3 && kShapes[s].CLS && kShapes[s].NWE == kShapes[v].NWE && kShapes[s].NG == kShapes[v].NG && kShapes[s].NJA == kShapes[v].NJA &&
                kShapes[s].NJB == kShapes[v].NJB && kShapes[s].HS == kShapes[v].HS)
                v_lo = s;
    p.n_cls = v_lo >= 0 ? 2 : 1;
    p.cls_xk = (float)(2.0 * 3.0 * szm / std::sqrt(2.0) / 0.95);
    p.cls_ylim = (float)(0.5 * gr.n_y * px);
    p.cls_tol = 2e-5f;
    const Shape& c = kShapes[v];
    const int n_regions = 1 + c.NG;
    p.nr_min = nr_lo; p.nr_max = nr_hi;
    p.HS = c.HS;
    p.Sy = std::max(1, p.HS - 2 * p.Hy);
    // shared memory: w region + accumulator regions + task table.  The sub-tile width Sz (8 or 4 columns) is the
    // one that lets most warps live on an SM (228 KB per SM, 1 KB reserved per CTA, 227 KB per CTA); 8 on a tie.
    const size_t budget = 225 * 1024, sm_bytes = 228 * 1024, tab_bytes = tab.size() * sizeof(uint32_t);
    const int cta_warps = c.NWE * c.NG;
    size_t smem = 0;
    {
        int best_sz = g_opt.sz > 0 ? (int)g_opt.sz : 4;      // a forced width is never replaced: if its regions do not fit,
        size_t best_warps = 0;                                //  smem > budget below sends every event to the direct kernel
        for (int sz : {8, 4}) {
            if (g_opt.sz > 0) sz = (int)g_opt.sz;
            const size_t need = n_regions * sizeof(float) * (size_t)p.HS * (sz + 2 * p.Hz) + tab_bytes;
            const size_t ctas = need <= budget ? std::min<size_t>(sm_bytes / (need + 2048), 2048 / (32 * cta_warps)) : 0;
            if (ctas * cta_warps > best_warps) { best_warps = ctas * cta_warps; best_sz = sz; }
        }
        p.Sz = best_sz;
        p.WZ = p.Sz + 2 * p.Hz;
        smem = n_regions * sizeof(float) * (size_t)p.HS * p.WZ + tab_bytes;
    }
    if (smem > budget || !tiles_ok || p.WZ < c.NJA + 4 || g_opt.force_direct || g_opt.exact_kernel > 0) {
        p.t_max = -1.f; smem = 0; p.nr_min = p.nr_max = 0; tab.clear();
        p.n_cls = 1; v_lo = -1;
    }
    p.nby = (gr.n_y + 2 * p.Hy + p.Sy - 1) / p.Sy;
    p.nbz = (gr.n_z + 2 * p.Hz + p.Sz - 1) / p.Sz;
    // events per work item (one staging of w and one flush of the accumulator regions per item): measured on B200 with 10^7
    // events per launch - 256 events per group for the one-warp groups (config 3: 6.28 -> 6.21 ms against 128), 512 for the
    // multi-warp groups (config 5: 34.36 -> 33.99 ms, config 4: 24.64 -> 24.34 ms against 256); batch_chunk halves it for
    // small batches
    p.chunk = g_opt.chunk > 0 ? (int)g_opt.chunk : (c.NWE > 1 ? 512 : 256) * c.NG;
    out->dp = p;
    out->shape = v;
    out->shape_lo = v_lo;
    out->smem = smem;
    out->vs = eta != 0.0;
    if (tab_out) tab_out->swap(tab);
}

bool same_problem(const Workspace& w, const jpet_geometry& g, const jpet_grid& gr) {
    return w.s_valid && w.geom.R == g.R && w.geom.L == g.L && w.grid.n_y == gr.n_y && w.grid.n_z == gr.n_z && w.grid.pixel == gr.pixel;
}

int grid_for(int64_t M) { return (int)((M + 255) / 256); }

int ensure_binset(Workspace& w, BinSet& bs, int64_t n, bool need_sorted) {
    const DevParams& dp = w.plan.dp;
    size_t items_cap = (size_t)(n / batch_chunk(w, n)) + (size_t)dp.nby * dp.nbz * dp.n_cls + 2;
    const size_t need_floats = 16 * (size_t)std::max<int64_t>(n, 1);
    if (need_sorted && need_floats > bs.cap_events) {          // cap_events counts floats
        if (bs.owns_sorted) cudaFree(bs.sorted);
        bs.sorted = nullptr; bs.cap_events = 0;
        CUDA_TRY(cudaMalloc(&bs.sorted, sizeof(float) * need_floats));
        bs.cap_events = need_floats;
        bs.owns_sorted = true;
    }
    if (items_cap > bs.cap_items) {
        cudaFree(bs.items);
        bs.items = nullptr; bs.cap_items = 0;
        CUDA_TRY(cudaMalloc(&bs.items, sizeof(jpet::WorkItem) * items_cap));
        bs.cap_items = items_cap;
    }
    if (!bs.meta) CUDA_TRY(cudaMalloc(&bs.meta, jpet::kMetaWords * sizeof(int)));
    return JPET_OK;
}

void free_binset(BinSet& bs) {
    if (bs.owns_sorted) cudaFree(bs.sorted);
    cudaFree(bs.items);
    cudaFree(bs.meta);
    bs = BinSet{};
}

constexpr size_t kTileBytes = sizeof(float) * 3 * jpet::kBinTile;

int ensure_sort_attr(Workspace& w) {
    if (w.sort_attr_set) return JPET_OK;
    const int bytes = (int)(kTileBytes + sizeof(int) * jpet::kBinSmemMax);
    CUDA_TRY(cudaFuncSetAttribute(jpet::bin_count_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    CUDA_TRY(cudaFuncSetAttribute(jpet::bin_scatter_rec_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    w.sort_attr_set = true;
    return JPET_OK;
}

// Counting sort of one batch (<= kMaxBatch events) by sub-tile into bs.sorted, and its work items.
int bin_batch(Workspace& w, const float* events, int64_t n, BinSet& bs, cudaStream_t st) {
    const DevParams& dp = w.plan.dp;
    const int nb0 = dp.nby * dp.nbz, nb = nb0 * dp.n_cls;      // regular bins: of degree class 0, of all classes
    int rc = ensure_sort_attr(w);
    if (rc) return rc;
    if ((size_t)n > w.cap_place) {
        cudaFree(w.place);
        w.place = nullptr; w.cap_place = 0;
        CUDA_TRY(cudaMalloc(&w.place, sizeof(int2) * (size_t)n));
        w.cap_place = (size_t)n;
    }
    if ((size_t)(2 * (nb + 1)) > w.cap_counts) {
        cudaFree(w.counts);
        w.counts = nullptr; w.cap_counts = 0;
        CUDA_TRY(cudaMalloc(&w.counts, sizeof(int) * 2 * (size_t)(nb + 1)));
        w.cap_counts = (size_t)(2 * (nb + 1));
        w.counts_clean_nb = -1;
    }
    int* counts = w.counts;
    int* cursors = w.counts + (nb + 1);
    if (w.counts_clean_nb != nb) {        // bin_scan_kernel leaves the counts zeroed: a memset only when the layout changes
        CUDA_TRY(cudaMemsetAsync(counts, 0, sizeof(int) * (nb + 1), st));
        w.counts_clean_nb = nb;
    }
    const int blocks = (int)((n + jpet::kBinTile - 1) / jpet::kBinTile);
    const int use_smem = nb + 1 <= jpet::kBinSmemMax;
    const size_t smem_bytes = kTileBytes + (use_smem ? sizeof(int) * (size_t)(nb + 1) : 0);
    const int saved_clean = w.counts_clean_nb;
    w.counts_clean_nb = -1;                 // dirty until bin_scan_kernel has been queued (an error in between leaves it so)
    if (n > 0) {
        CUDA_TRY(launch_pdl(jpet::bin_count_kernel, dim3(blocks), dim3(jpet::kBinBlock), smem_bytes, st, events, (int)n, dp, w.place,
                            counts, nb + 1, use_smem));
        g_launches++;
    }
    CUDA_TRY(launch_pdl(jpet::bin_scan_kernel, dim3(1), dim3(1024), 0, st, counts, cursors, bs.items, bs.meta, nb, nb0, batch_chunk(w, n)));
    g_launches++;
    w.counts_clean_nb = saved_clean;
    if (n > 0) {
        CUDA_TRY(launch_pdl(jpet::bin_scatter_rec_kernel, dim3(blocks), dim3(jpet::kBinBlock), smem_bytes, st, events, (int)n,
                            (const int2*)w.place, cursors, reinterpret_cast<jpet::EventRec*>(bs.sorted), dp, nb + 1, use_smem));
        g_launches++;
    }
    CUDA_TRY(cudaGetLastError());
    bs.n = n;
    return JPET_OK;
}

int do_begin(Workspace& w, const jpet_geometry* g, const jpet_sigmas* sg, const jpet_grid* gr, const float* rho_in, cudaStream_t st) {
    int rc = validate(g, sg, gr);
    if (rc) return rc;
    if (!sg) return fail(JPET_E_INVAL, "NULL sigmas");
    if (!rho_in) return fail(JPET_E_INVAL, "NULL rho_in");
    const int M = gr->n_y * gr->n_z;
    if ((rc = ensure_images(w, M))) return rc;
    w.open = false;
    if (!same_problem(w, *g, *gr)) {
        jpet::sensitivity_kernel<<<grid_for(M), 256, 0, st>>>(w.s, gr->n_y, gr->n_z, gr->pixel, g->R, g->L);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
        w.geom = *g; w.grid = *gr; w.s_valid = true;
    }
    w.sig = *sg; w.M = M;
    {   // the plan depends only on these inputs: rebuild it (and the task table) when one of them changes
        PlanKey key;
        key.g = *g; key.sg = *sg; key.gr = *gr; key.a3 = g_opt.a3_coef; key.gamma = g_opt.gamma; key.sz_eta = g_opt.sz_eta;
        key.variant = g_opt.variant; key.sz = g_opt.sz; key.chunk = g_opt.chunk; key.force_direct = g_opt.force_direct;
        key.poly_off = g_opt.poly_off; key.exact = g_opt.exact_kernel; key.cls_off = g_opt.cls_off;
        if (!w.plan_valid || !(key == w.plan_key)) {
            make_plan(*g, *sg, *gr, &w.plan, &w.tab_host);
            w.plan_key = key;
            w.plan_valid = true;
        }
    }
    if (w.plan.shape < 0 || w.plan.shape >= kNumShapes) return fail(JPET_E_INVAL, "unknown kernel shape");
    if (!w.tab_host.empty() && w.tab_host != w.tab_uploaded) {        // task table of the tiled event kernel
        if (w.tab_host.size() > w.cap_tab) {
            cudaFree(w.tab);
            w.tab = nullptr; w.cap_tab = 0;
            CUDA_TRY(cudaMalloc(&w.tab, sizeof(uint32_t) * w.tab_host.size()));
            w.cap_tab = w.tab_host.size();
        }
        w.tab_uploaded = w.tab_host;      // the copy below reads tab_uploaded, which stays put until the next change
        CUDA_TRY(cudaMemcpyAsync(w.tab, w.tab_uploaded.data(), sizeof(uint32_t) * w.tab_uploaded.size(), cudaMemcpyHostToDevice, st));
    }
    w.tk_used = 0;                 // last_kernel_ns covers the event-kernel launches of one iteration
    CUDA_TRY(launch_pdl(jpet::prepass_kernel, dim3(grid_for(M)), dim3(256), 0, st, (const float*)w.s, rho_in, w.wT, w.accT, gr->n_y,
                        gr->n_z, w.counters));
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    w.open = true;
    return JPET_OK;
}

int do_accumulate(Workspace& w, const float* events, int64_t n, cudaStream_t st) {
    if (!w.open) return fail(JPET_E_INVAL, "jpet_mlem_accumulate without jpet_mlem_begin");
    if (n < 0) return fail(JPET_E_INVAL, "n < 0");
    if (n > 0 && !events) return fail(JPET_E_INVAL, "NULL events");
    for (int64_t off = 0; off < n; off += kMaxBatch) {
        int64_t nb = std::min(kMaxBatch, n - off);
        int rc = ensure_binset(w, w.scratch, nb, true);
        if (!rc) rc = bin_batch(w, events + 3 * off, nb, w.scratch, st);
        if (!rc) rc = run_binset(w, w.scratch, st);
        if (rc) { w.open = false; return rc; }
    }
    return JPET_OK;
}

int do_end(Workspace& w, const float* rho_in, float* rho_out, const float* const* peers, int n_peers, cudaStream_t st) {
    if (!w.open) return fail(JPET_E_INVAL, "jpet_mlem_end without jpet_mlem_begin");
    if (!rho_in || !rho_out) return fail(JPET_E_INVAL, "NULL image pointer");
    jpet::PeerAcc pa{};
    if (peers) {
        if (n_peers < 1 || n_peers > jpet::kMaxPeers) return fail(JPET_E_INVAL, "n_peers must be 1 .. %d", jpet::kMaxPeers);
        for (int q = 0; q < n_peers; ++q) {
            if (!peers[q]) return fail(JPET_E_INVAL, "NULL peer accumulator");
            pa.acc[q] = peers[q];
        }
        pa.n = n_peers;
    } else {
        pa.acc[0] = w.accT;
        pa.n = 1;
    }
    w.open = false;
    CUDA_TRY(launch_pdl(jpet::finalise_kernel, dim3(grid_for(w.M)), dim3(256), 0, st, (const float*)w.s, rho_in, pa, rho_out, w.grid.n_y,
                        w.grid.n_z));
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

// n_iter iterations over device-resident events; the events are binned once (first iteration) and the
// sorted copy is reused by the others (events never change between iterations).
int iterate_many(Workspace& w, const float* events, int64_t n, const jpet_geometry* g, const jpet_sigmas* sg, const jpet_grid* gr,
                 const float* rho_start, float* rho_out, int n_iter, cudaStream_t st) {
    const float* cur = rho_start;
    const int64_t n_batches = (n + kMaxBatch - 1) / kMaxBatch;
    const bool keep = n_iter > 1;
    if (keep) while ((int64_t)w.kept.size() < n_batches) w.kept.emplace_back();
    for (int it = 0; it < n_iter; ++it) {
        float* nxt = (it == n_iter - 1) ? rho_out : (cur == w.rho_a ? w.rho_b : w.rho_a);
        int rc = do_begin(w, g, sg, gr, cur, st);        // fixes the plan (kernel shape, tiling) for this problem
        if (rc) return rc;
        if (keep && it == 0 && 16 * (size_t)n > w.cap_kept_sorted) {      // capacity counts floats
            cudaFree(w.kept_sorted);
            w.kept_sorted = nullptr; w.cap_kept_sorted = 0;
            cudaError_t e = cudaMalloc(&w.kept_sorted, sizeof(float) * 16 * (size_t)n);
            if (e != cudaSuccess) { w.open = false; return fail(JPET_E_CUDA, "cudaMalloc of the kept records failed: %s", cudaGetErrorString(e)); }
            w.cap_kept_sorted = 16 * (size_t)n;
        }
        if (!keep) {
            if ((rc = do_accumulate(w, events, n, st))) return rc;
        } else {
            for (int64_t b = 0; b < n_batches; ++b) {
                BinSet& bs = w.kept[b];
                int64_t off = b * kMaxBatch, nb = std::min(kMaxBatch, n - off);
                if (it == 0) {
                    if (bs.owns_sorted) cudaFree(bs.sorted);
                    bs.owns_sorted = false;
                    bs.sorted = w.kept_sorted + 16 * (size_t)off;
                    rc = ensure_binset(w, bs, nb, false);
                    if (!rc) rc = bin_batch(w, events + 3 * off, nb, bs, st);
                }
                if (!rc) rc = run_binset(w, bs, st);
                if (rc) { w.open = false; return rc; }
            }
        }
        if ((rc = do_end(w, cur, nxt, nullptr, 0, st))) return rc;
        cur = nxt;
    }
    return JPET_OK;
}

int ensure_host_path(Workspace& w, size_t stage_bytes) {
    if (!w.copy_stream) {
        CUDA_TRY(cudaStreamCreateWithFlags(&w.copy_stream, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&w.compute_stream, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CUDA_TRY(cudaEventCreateWithFlags(&w.ev_copy[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&w.ev_done[i], cudaEventDisableTiming));
        }
    }
    if (stage_bytes > w.cap_stage) {
        cudaFree(w.stage);
        w.stage = nullptr;
        w.cap_stage = 0;
        CUDA_TRY(cudaMalloc(&w.stage, stage_bytes));
        w.cap_stage = stage_bytes;
    }
    return JPET_OK;
}

// One iteration's accumulate phase from host events.  If everything fits the staging buffer it is filled chunk by chunk
// (copy of chunk c+1 overlaps compute of chunk c) and left resident; otherwise two chunk-sized slots are used as a
// ring: before a slot is overwritten the copy stream waits for the kernels that read its previous content - also across
// iterations (slot_used lives in the workspace, not in this call).
int accumulate_from_host(Workspace& w, const float* events_host, int64_t n, int64_t chunk, bool fits) {
    cudaStream_t cs = w.copy_stream, ks = w.compute_stream;
    if (fits) {
        // resident events: upload and compute in batches that double from `chunk` up to the batch size of the device path -
        // the first batch starts after one chunk has arrived, every later upload hides behind the previous batch's kernels,
        // and most events are sorted and walked in full-size batches (config 5 through 2x10^6-event batches: 369 ms per
        // iteration, 5 % over the device-resident 349 ms - five times as many partly filled work items)
        int b = 0;
        int64_t batch = chunk;
        for (int64_t off = 0; off < n; ++b) {
            const int64_t nb = std::min(batch, n - off);
            float* dst = w.stage + 3 * off;
            CUDA_TRY(cudaMemcpyAsync(dst, events_host + 3 * off, sizeof(float) * 3 * nb, cudaMemcpyHostToDevice, cs));
            CUDA_TRY(cudaEventRecord(w.ev_copy[b & 1], cs));
            CUDA_TRY(cudaStreamWaitEvent(ks, w.ev_copy[b & 1], 0));
            int rc = do_accumulate(w, dst, nb, ks);
            if (rc) return rc;
            off += nb;
            batch = std::min<int64_t>(2 * batch, kMaxBatch);
        }
        return JPET_OK;
    }
    int c = 0;
    for (int64_t off = 0; off < n; off += chunk, ++c) {
        int64_t nb = std::min(chunk, n - off);
        int slot = c & 1;
        float* dst = fits ? w.stage + 3 * off : w.stage + 3 * (int64_t)slot * chunk;
        if (!fits && w.slot_used[slot]) CUDA_TRY(cudaStreamWaitEvent(cs, w.ev_done[slot], 0));   // slot free again
        CUDA_TRY(cudaMemcpyAsync(dst, events_host + 3 * off, sizeof(float) * 3 * nb, cudaMemcpyHostToDevice, cs));
        CUDA_TRY(cudaEventRecord(w.ev_copy[slot], cs));
        CUDA_TRY(cudaStreamWaitEvent(ks, w.ev_copy[slot], 0));
        int rc = do_accumulate(w, dst, nb, ks);
        if (rc) return rc;
        if (!fits) { CUDA_TRY(cudaEventRecord(w.ev_done[slot], ks)); w.slot_used[slot] = true; }
    }
    return JPET_OK;
}

int reconstruct_host_impl(const float* events_host, int64_t n, const jpet_geometry* g, const jpet_sigmas* sg,
                          const jpet_grid* gr, const float* rho_init_host, float* rho_out_host, int32_t n_iter, int64_t chunk) {
    int rc = validate(g, sg, gr);
    if (rc) return rc;
    if (!sg) return fail(JPET_E_INVAL, "NULL sigmas");
    if (n < 0 || n_iter < 0) return fail(JPET_E_INVAL, "n < 0 or n_iter < 0");
    if ((n > 0 && !events_host) || !rho_out_host) return fail(JPET_E_INVAL, "NULL host pointer");
    Workspace* wp = nullptr;
    if ((rc = current_ws(&wp))) return rc;
    Workspace& w = *wp;
    const int M = gr->n_y * gr->n_z;
    if ((rc = ensure_images(w, M))) return rc;
    // upload chunk: a quarter of the events, between 5x10^5 and 2x10^6, so that the copy of chunk c+1 overlaps the sort
    // and the event kernel of chunk c also for one-batch problems (config 2 on a box with a 12 GB/s host link:
    // 1.6 ms with one chunk, 1.07 ms with two; no difference on a 50 GB/s link)
    if (chunk <= 0) chunk = std::min<int64_t>(2000000, std::max<int64_t>(500000, (n + 3) / 4));
    chunk = std::min<int64_t>(chunk, std::max<int64_t>(n, 1));
    const int64_t budget = g_opt.stage_bytes > 0 ? g_opt.stage_bytes : kStageDefault;
    const bool fits = (int64_t)sizeof(float) * 3 * n <= budget;
    size_t stage_bytes = fits ? sizeof(float) * 3 * (size_t)std::max<int64_t>(n, 1) : sizeof(float) * 3 * 2 * (size_t)chunk;
    if ((rc = ensure_host_path(w, stage_bytes))) return rc;
    cudaStream_t ks = w.compute_stream;
    if ((rc = enter(w, ks))) return rc;
    CallScope scope(w, ks, true);
    w.slot_used[0] = w.slot_used[1] = false;       // nothing of an earlier call is in flight: every host call ends synchronised
                                                   // on both internal streams, error returns included (CallScope)
    float* cur = w.rho_a;
    float* nxt = w.rho_b;
    if (rho_init_host) {
        CUDA_TRY(cudaMemcpyAsync(cur, rho_init_host, sizeof(float) * M, cudaMemcpyHostToDevice, ks));
    } else {
        jpet::ones_kernel<<<grid_for(M), 256, 0, ks>>>(cur, M);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
    }
    if (n_iter > 0) {
        // first iteration: the upload of chunk c+1 overlaps the binning + event kernels of chunk c
        if ((rc = do_begin(w, g, sg, gr, cur, ks))) return rc;
        if ((rc = accumulate_from_host(w, events_host, n, chunk, fits))) return rc;
        if ((rc = do_end(w, cur, nxt, nullptr, 0, ks))) return rc;
        std::swap(cur, nxt);
        if (n_iter > 1) {
            if (fits) {         // events are now resident in the staging buffer: bin once, iterate
                if ((rc = iterate_many(w, w.stage, n, g, sg, gr, cur, nxt, n_iter - 1, ks))) return rc;
                std::swap(cur, nxt);
            } else {
                for (int it = 1; it < n_iter; ++it) {
                    if ((rc = do_begin(w, g, sg, gr, cur, ks))) return rc;
                    if ((rc = accumulate_from_host(w, events_host, n, chunk, false))) return rc;
                    if ((rc = do_end(w, cur, nxt, nullptr, 0, ks))) return rc;
                    std::swap(cur, nxt);
                }
            }
        }
    }
    CUDA_TRY(cudaMemcpyAsync(rho_out_host, cur, sizeof(float) * M, cudaMemcpyDeviceToHost, ks));
    return scope.finish();
}

void release_ws(Workspace& w) {
    cudaFree(w.s); cudaFree(w.wT); cudaFree(w.accT); cudaFree(w.rho_a); cudaFree(w.rho_b);
    cudaFree(w.counters); cudaFree(w.stage); cudaFree(w.place); cudaFree(w.counts); cudaFree(w.kept_sorted);
    cudaFree(w.tab);
    free_binset(w.scratch);
    for (auto& bs : w.kept) free_binset(bs);
    for (int i = 0; i < 2; ++i) {
        if (w.ev_copy[i]) cudaEventDestroy(w.ev_copy[i]);
        if (w.ev_done[i]) cudaEventDestroy(w.ev_done[i]);
    }
    if (w.ev_last) cudaEventDestroy(w.ev_last);
    for (cudaEvent_t e : w.tk)
        if (e) cudaEventDestroy(e);
    if (w.copy_stream) cudaStreamDestroy(w.copy_stream);
    if (w.compute_stream) cudaStreamDestroy(w.compute_stream);
}

// ---- jpet_mlem_iterate_noalloc: one iteration whose scratch is a fixed array inside the library image ------------------
// Some users of this library must not, or cannot, allocate device memory at the moment they need an iteration: an
// acquisition or monitoring loop with a latency budget (cudaMalloc / cudaFree stall every stream of the device while they
// run), a plug-in inside a host program that has handed all of HBM to its own pool (cudaMalloc then simply fails), a
// process whose rules forbid driver allocations after start-up.  For them the three scratch images of an iteration
// (s of Eq. 4, w = s rho, the back-projection accumulator), the counters and the meta words of the direct event kernel
// live in the array below.  It is part of the loaded library: every GPU on which the library's kernels get loaded keeps
// its own 3 MiB copy until the process exits, whether or not the entry point is ever called.
constexpr int kNoAllocMaxPixels = JPET_NOALLOC_MAX_PIXELS;
constexpr size_t kNoAllocImageBytes = sizeof(float) * (size_t)kNoAllocMaxPixels;      // 1 MiB: keeps every part 256-aligned
constexpr size_t kNoAllocCountersAt = 3 * kNoAllocImageBytes;                          // 4 x unsigned long long
constexpr size_t kNoAllocMetaAt = kNoAllocCountersAt + 64;                             // kMetaWords x int
constexpr size_t kNoAllocBytes = kNoAllocCountersAt + 256;
static_assert(kNoAllocMetaAt + sizeof(int) * jpet::kMetaWords <= kNoAllocBytes, "scratch tail too small");
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

// In host code `g_noalloc_scratch` is only a handle for the runtime, not an address a kernel could use: the device
// address is asked for once per device, with that device current, and remembered.
struct NoAllocDevice { unsigned char* base = nullptr; int sm_count = 0; };
std::map<int, NoAllocDevice> g_noalloc_dev;

int noalloc_device(NoAllocDevice* out) {
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    auto it = g_noalloc_dev.find(dev);
    if (it == g_noalloc_dev.end()) {
        NoAllocDevice d;
        void* ptr = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&ptr, g_noalloc_scratch));
        if (!ptr) return fail(JPET_E_CUDA, "cudaGetSymbolAddress gave no address for the static scratch on device %d", dev);
        d.base = static_cast<unsigned char*>(ptr);
        CUDA_TRY(cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev));
        it = g_noalloc_dev.emplace(dev, d).first;
    }
    *out = it->second;
    return JPET_OK;
}

// meta words of a "sorted batch" that is simply the caller's event array: the direct bin is all of it
__global__ void noalloc_meta_kernel(int* __restrict__ meta, int n) {
    const int i = threadIdx.x;
    if (i < jpet::kMetaWords) meta[i] = i == jpet::kMetaDirectCount ? n : 0;
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
    int rc = validate(geometry, sigmas, grid);
    if (rc) return rc;
    Workspace* w = nullptr;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = current_ws(&w)) || (rc = enter(*w, st))) return rc;
    CallScope scope(*w, st);
    if ((rc = do_begin(*w, geometry, sigmas, grid, rho_in_dev, st))) return rc;
    return scope.finish();
}

int jpet_mlem_accumulate(const float* events_dev, int64_t n_batch, void* cuda_stream) {
    g_err.clear();
    Workspace* w = device_ws();
    if (!w || !w->open) return fail(JPET_E_INVAL, "jpet_mlem_accumulate without jpet_mlem_begin");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = enter(*w, st);
    if (rc) return rc;
    CallScope scope(*w, st);
    if ((rc = do_accumulate(*w, events_dev, n_batch, st))) return rc;
    return scope.finish();
}

int jpet_mlem_end(const float* rho_in_dev, float* rho_out_dev, void* cuda_stream) {
    g_err.clear();
    Workspace* w = device_ws();
    if (!w || !w->open) return fail(JPET_E_INVAL, "jpet_mlem_end without jpet_mlem_begin");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = enter(*w, st);
    if (rc) return rc;
    CallScope scope(*w, st);
    if ((rc = do_end(*w, rho_in_dev, rho_out_dev, nullptr, 0, st))) return rc;
    return scope.finish();
}

int jpet_mlem_end_peers(const float* rho_in_dev, float* rho_out_dev, const float* const* peer_acc_dev, int32_t n_peers,
                        void* cuda_stream) {
    g_err.clear();
    Workspace* w = device_ws();
    if (!w || !w->open) return fail(JPET_E_INVAL, "jpet_mlem_end_peers without jpet_mlem_begin");
    if (!peer_acc_dev) return fail(JPET_E_INVAL, "NULL peer list");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = enter(*w, st);
    if (rc) return rc;
    CallScope scope(*w, st);
    if ((rc = do_end(*w, rho_in_dev, rho_out_dev, peer_acc_dev, n_peers, st))) return rc;
    return scope.finish();
}

int jpet_mlem_accumulator(float** acc_dev, int64_t* n_floats) {
    g_err.clear();
    Workspace* w = device_ws();
    if (!w || !w->open) return fail(JPET_E_INVAL, "jpet_mlem_accumulator without an open iteration (jpet_mlem_begin)");
    if (!acc_dev || !n_floats) return fail(JPET_E_INVAL, "NULL output pointer");
    *acc_dev = w->accT;
    *n_floats = w->M;
    return JPET_OK;
}

int jpet_ipc_export(const void* dev_ptr, void* handle64_out) {
    g_err.clear();
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "cudaIpcMemHandle_t is 64 bytes");
    if (!dev_ptr || !handle64_out) return fail(JPET_E_INVAL, "NULL pointer");
    cudaIpcMemHandle_t h;
    CUDA_TRY(cudaIpcGetMemHandle(&h, const_cast<void*>(dev_ptr)));
    memcpy(handle64_out, &h, sizeof h);
    return JPET_OK;
}

int jpet_ipc_open(const void* handle64, void** dev_ptr_out) {
    g_err.clear();
    if (!handle64 || !dev_ptr_out) return fail(JPET_E_INVAL, "NULL pointer");
    cudaIpcMemHandle_t h;
    memcpy(&h, handle64, sizeof h);
    CUDA_TRY(cudaIpcOpenMemHandle(dev_ptr_out, h, cudaIpcMemLazyEnablePeerAccess));
    return JPET_OK;
}

int jpet_ipc_close(void* dev_ptr) {
    g_err.clear();
    if (!dev_ptr) return fail(JPET_E_INVAL, "NULL pointer");
    CUDA_TRY(cudaIpcCloseMemHandle(dev_ptr));
    return JPET_OK;
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
    Workspace* w = nullptr;
    if ((rc = current_ws(&w)) || (rc = enter(*w, st))) return rc;
    CallScope scope(*w, st);
    if ((rc = do_begin(*w, geometry, sigmas, grid, rho_in_dev, st))) return rc;
    if ((rc = do_accumulate(*w, events_dev, n, st))) return rc;
    if ((rc = do_end(*w, rho_in_dev, rho_out_dev, nullptr, 0, st))) return rc;
    return scope.finish();
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
    cudaStream_t st = (cudaStream_t)cuda_stream;
    Workspace* w = nullptr;
    if ((rc = current_ws(&w)) || (rc = enter(*w, st))) return rc;
    CallScope scope(*w, st);
    const int M = grid->n_y * grid->n_z;
    if ((rc = ensure_images(*w, M))) return rc;
    // ping-pong through the workspace so that rho_out may alias rho_init and is written once per iteration
    const float* cur = rho_init_dev;
    if (!cur) {
        jpet::ones_kernel<<<grid_for(M), 256, 0, st>>>(w->rho_a, M);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
        cur = w->rho_a;
    }
    if (n_iter == 0) {
        if (cur != rho_out_dev) CUDA_TRY(cudaMemcpyAsync(rho_out_dev, cur, sizeof(float) * M, cudaMemcpyDeviceToDevice, st));
        return scope.finish();
    }
    if ((rc = iterate_many(*w, events_dev, n, geometry, sigmas, grid, cur, rho_out_dev, n_iter, st))) return rc;
    return scope.finish();
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
    Workspace* w = device_ws();
    if (!w || !w->counters) return fail(JPET_E_INVAL, "no iteration has been run");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int rc = enter(*w, st);
    if (rc) return rc;
    unsigned long long h[3];
    CUDA_TRY(cudaMemcpyAsync(h, w->counters, sizeof h, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (n_evals_host) *n_evals_host = h[0];
    if (n_skipped_host) *n_skipped_host = h[1];
    if (h[2]) return fail(JPET_E_INTERNAL, "the event kernel met %llu records it could not hold (piece longer than its register slot or "
                          "row count outside the task table): the image of this iteration is incomplete", h[2]);
    return JPET_OK;
}

int jpet_count_evals(const float* events_dev, int64_t n, const jpet_geometry* geometry, const jpet_sigmas* sigmas,
                     const jpet_grid* grid, uint64_t* n_evals_host, uint64_t* n_skipped_host, void* cuda_stream) {
    g_err.clear();
    int rc = validate(geometry, sigmas, grid);
    if (rc) return rc;
    if (!sigmas) return fail(JPET_E_INVAL, "NULL sigmas");
    if (n < 0 || (n > 0 && !events_dev)) return fail(JPET_E_INVAL, "bad events");
    Workspace* w = nullptr;
    if ((rc = current_ws(&w))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unsigned long long* d = nullptr;
    CUDA_TRY(cudaMalloc(&d, 2 * sizeof(unsigned long long)));
    cudaError_t e = cudaMemsetAsync(d, 0, 2 * sizeof(unsigned long long), st);
    jpet_host::RowsPlan plan;
    make_plan(*geometry, *sigmas, *grid, &plan);
    if (e == cudaSuccess && n > 0) {
        int blocks = (int)std::min<int64_t>((n + 255) / 256, (int64_t)w->sm_count * 8);
        jpet::count_evals_kernel<<<blocks, 256, 0, st>>>(events_dev, (long long)n, plan.dp, d);
        g_launches++;
    }
    unsigned long long h[2] = {0, 0};
    if (e == cudaSuccess) e = cudaMemcpyAsync(h, d, sizeof h, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d);
    if (e != cudaSuccess) return fail(JPET_E_CUDA, "count_evals: %s", cudaGetErrorString(e));
    if (n_evals_host) *n_evals_host = h[0];
    if (n_skipped_host) *n_skipped_host = h[1];
    return JPET_OK;
}

int jpet_direct_histogram(const float* events_dev, int64_t n, const jpet_geometry* geometry, const jpet_grid* grid,
                          uint32_t* hist_dev, uint64_t* n_outside_host, void* cuda_stream) {
    g_err.clear();
    int rc = validate(geometry, nullptr, grid);
    if (rc) return rc;
    if (n < 0 || (n > 0 && !events_dev)) return fail(JPET_E_INVAL, "bad events");
    if (n > 0x7fffffffll) return fail(JPET_E_INVAL, "at most 2^31 - 1 events per call");
    if (!hist_dev) return fail(JPET_E_INVAL, "NULL hist_dev");
    Workspace* w = nullptr;
    if ((rc = current_ws(&w))) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = enter(*w, st))) return rc;
    CallScope scope(*w, st);
    if (!w->counters) CUDA_TRY(cudaMalloc(&w->counters, 4 * sizeof(unsigned long long)));
    CUDA_TRY(cudaMemsetAsync(w->counters + 3, 0, sizeof(unsigned long long), st));
    jpet::HistParams h;
    h.n_y = grid->n_y; h.n_z = grid->n_z;
    h.inv2R = (float)(1.0 / (2.0 * (double)geometry->R));
    h.inv_px = (float)(1.0 / (double)grid->pixel);
    h.oy = (float)(0.5 * (grid->n_y - 1) + 0.5);
    h.oz = (float)(0.5 * (grid->n_z - 1) + 0.5);
    // at most 2^30 events per launch: the kernel walks its tiles with 32-bit offsets, and with one tile per block the stride
    // is about the launch size (base + stride < 2^31); 2^30 events keep every launch's first event 16-byte aligned
    constexpr int64_t kHistMaxLaunch = 1ll << 30;
    const int M = grid->n_y * grid->n_z;
    const int use_smem = M <= jpet::kHistSmemMax;
    const size_t smem = kTileBytes + (use_smem ? sizeof(unsigned int) * (size_t)M : 0);
    for (int64_t off = 0; off < n; off += kHistMaxLaunch) {
        const int64_t nl = std::min<int64_t>(kHistMaxLaunch, n - off);
        const int tiles = (int)((nl + jpet::kBinTile - 1) / jpet::kBinTile);
        // shared-memory histograms: a persistent grid (one flush per block); global atomics: one tile per block
        const int blocks = use_smem ? std::min(tiles, w->sm_count * 4) : tiles;
        jpet::direct_histogram_kernel<<<blocks, jpet::kBinBlock, smem, st>>>(events_dev + 3 * off, (int)nl, h, hist_dev, w->counters + 3, use_smem);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
    }
    if ((rc = scope.finish())) return rc;
    if (n_outside_host) {
        unsigned long long out = 0;
        CUDA_TRY(cudaMemcpyAsync(&out, w->counters + 3, sizeof out, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        *n_outside_host = out;
    }
    return JPET_OK;
}

int jpet_generate_events(const jpet_primitive* phantom_host, int32_t n_primitives, int64_t n, int64_t first,
                         const jpet_geometry* geometry, const jpet_sigmas* sigmas, uint64_t seed, float* events_dev,
                         void* cuda_stream) {
    g_err.clear();
    if (!geometry || !sigmas) return fail(JPET_E_INVAL, "NULL geometry or sigmas");
    if (!(geometry->R > 0.f) || !(geometry->L > 0.f) || !std::isfinite(geometry->R) || !std::isfinite(geometry->L))
        return fail(JPET_E_INVAL, "R and L must be positive and finite");
    if (!(sigmas->sigma_z >= 0.f) || !(sigmas->sigma_dl >= 0.f) || !std::isfinite(sigmas->sigma_z) || !std::isfinite(sigmas->sigma_dl))
        return fail(JPET_E_INVAL, "sigmas must be non-negative and finite");
    if (!phantom_host || n_primitives < 1 || n_primitives > jpet::kMaxPrimitives)
        return fail(JPET_E_INVAL, "the phantom must hold 1 .. %d primitives", jpet::kMaxPrimitives);
    if (n < 0 || first < 0 || (n > 0 && !events_dev)) return fail(JPET_E_INVAL, "bad n, first or events_dev");
    jpet::PhantomDev ph{};
    ph.n = n_primitives;
    double y0 = 1e300, y1 = -1e300, z0 = 1e300, z1 = -1e300, rho_max = 0.0;
    for (int k = 0; k < n_primitives; ++k) {
        const jpet_primitive& q = phantom_host[k];
        if ((q.kind != 0 && q.kind != 1) || !(q.hy > 0.f) || !(q.hz > 0.f) || !(q.intensity >= 0.f) || !std::isfinite(q.cy) ||
            !std::isfinite(q.cz) || !std::isfinite(q.hy) || !std::isfinite(q.hz) || !std::isfinite(q.phi_deg) || !std::isfinite(q.intensity))
            return fail(JPET_E_INVAL, "primitive %d: kind must be 0 or 1, half sizes positive, intensity >= 0, all finite", k);
        const double phi = (double)q.phi_deg * 3.14159265358979323846 / 180.0, c = std::cos(phi), s = std::sin(phi);
        double ey, ez;
        if (q.kind == 0) { ez = std::hypot(q.hz * c, q.hy * s); ey = std::hypot(q.hz * s, q.hy * c); }
        else { ez = q.hz * std::fabs(c) + q.hy * std::fabs(s); ey = q.hz * std::fabs(s) + q.hy * std::fabs(c); }
        y0 = std::min(y0, q.cy - ey); y1 = std::max(y1, q.cy + ey);
        z0 = std::min(z0, q.cz - ez); z1 = std::max(z1, q.cz + ez);
        rho_max = std::max(rho_max, (double)q.intensity);
        ph.kind[k] = q.kind; ph.cy[k] = q.cy; ph.cz[k] = q.cz;
        ph.inv_hy[k] = (float)(1.0 / q.hy); ph.inv_hz[k] = (float)(1.0 / q.hz);
        ph.cphi[k] = (float)c; ph.sphi[k] = (float)s;
    }
    if (!(rho_max > 0.0)) return fail(JPET_E_INVAL, "the phantom has no primitive with positive intensity");
    for (int k = 0; k < n_primitives; ++k) ph.rel[k] = (float)(phantom_host[k].intensity / rho_max);
    ph.y0 = (float)y0; ph.y1 = (float)y1; ph.z0 = (float)z0; ph.z1 = (float)z1;
    ph.R = geometry->R; ph.half_L = 0.5f * geometry->L; ph.sigma_z = sigmas->sigma_z; ph.sigma_dl = sigmas->sigma_dl;
    if (n == 0) return JPET_OK;
    Workspace* w = nullptr;
    int rc = current_ws(&w);
    if (rc) return rc;
    const int blocks = (int)std::min<int64_t>((n + 255) / 256, (int64_t)w->sm_count * 16);
    jpet::generate_events_kernel<<<blocks, 256, 0, (cudaStream_t)cuda_stream>>>(events_dev, (long long)n, (unsigned long long)first,
                                                                              (unsigned long long)seed, ph);
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

int jpet_set_a3_coef(float k) {
    g_err.clear();
    if (!std::isfinite(k)) return fail(JPET_E_INVAL, "a3 coefficient must be finite");
    g_opt.a3_coef = k;
    return JPET_OK;
}

float jpet_get_a3_coef(void) { return g_opt.a3_coef; }

int jpet_set_gamma(float gamma) {
    g_err.clear();
    if (!std::isfinite(gamma)) return fail(JPET_E_INVAL, "gamma must be finite");
    g_opt.gamma = gamma;
    return JPET_OK;
}

float jpet_get_gamma(void) { return g_opt.gamma; }

int jpet_set_sigma_z_edge(float eta) {
    g_err.clear();
    if (!(eta >= 0.f && eta <= 1.f)) return fail(JPET_E_INVAL, "the sigma_z edge coefficient must lie in [0, 1]");
    g_opt.sz_eta = eta;
    return JPET_OK;
}

float jpet_get_sigma_z_edge(void) { return g_opt.sz_eta; }

int jpet_set_option(const char* name, int64_t value) {
    g_err.clear();
    if (!name) return fail(JPET_E_INVAL, "NULL option name");
    if (!strcmp(name, "force_direct")) {
        if (value < 0 || value > 1) return fail(JPET_E_INVAL, "force_direct must be 0 or 1");
        g_opt.force_direct = value;
    } else if (!strcmp(name, "time_kernel")) {
        if (value < 0 || value > 1) return fail(JPET_E_INVAL, "time_kernel must be 0 or 1");
        g_opt.time_kernel = value;
        for (auto& kv : g_ctx) kv.second->tk_used = 0;
    } else if (!strcmp(name, "sub_tile_z")) {
        if (value < 0 || value > 256) return fail(JPET_E_INVAL, "sub_tile_z must be 0 (auto) .. 256");
        g_opt.sz = value;
    } else if (!strcmp(name, "chunk")) {
        if (value < 0 || value > (1 << 20)) return fail(JPET_E_INVAL, "chunk must be 0 (auto) .. 2^20");
        g_opt.chunk = value;
    } else if (!strcmp(name, "variant")) {
        if (value < -1 || value >= kNumShapes) return fail(JPET_E_INVAL, "variant must be -1 (auto) .. %d", kNumShapes - 1);
        g_opt.variant = value;
    } else if (!strcmp(name, "poly_off")) {
        g_opt.poly_off = value != 0;
    } else if (!strcmp(name, "degree_classes_off")) {
        g_opt.cls_off = value != 0;
    } else if (!strcmp(name, "pdl")) {
        g_opt.pdl = value != 0;
    } else if (!strcmp(name, "ctas_per_sm")) {
        if (value < 0 || value > 32) return fail(JPET_E_INVAL, "ctas_per_sm must be 0 (auto) .. 32");
        g_opt.ctas_per_sm = value;
    } else if (!strcmp(name, "stage_bytes")) {
        if (value < 0) return fail(JPET_E_INVAL, "stage_bytes must be >= 0 (0 = default)");
        g_opt.stage_bytes = value;
    } else if (!strcmp(name, "exact_kernel")) {
        if (value < 0 || value > 4096) return fail(JPET_E_INVAL, "exact_kernel must be 0 (off) .. 4096 quadrature nodes");
        g_opt.exact_kernel = value;
    } else {
        return fail(JPET_E_INVAL, "unknown option '%s'", name);
    }
    return JPET_OK;
}

int64_t jpet_get_option(const char* name) {
    if (!name) return -1;
    if (!strcmp(name, "force_direct")) return g_opt.force_direct;
    if (!strcmp(name, "chunk")) return g_opt.chunk;
    if (!strcmp(name, "sub_tile_z")) return g_opt.sz;
    if (!strcmp(name, "time_kernel")) return g_opt.time_kernel;
    if (!strcmp(name, "variant")) return g_opt.variant;
    if (!strcmp(name, "poly_off")) return g_opt.poly_off;
    if (!strcmp(name, "degree_classes_off")) return g_opt.cls_off;
    if (!strcmp(name, "pdl")) return g_opt.pdl;
    if (!strcmp(name, "ctas_per_sm")) return g_opt.ctas_per_sm;
    if (!strcmp(name, "stage_bytes")) return g_opt.stage_bytes;
    if (!strcmp(name, "exact_kernel")) return g_opt.exact_kernel;
    Workspace* w = last_ws();
    if (!w) return -1;
    if (!strcmp(name, "last_kernel_ns")) {      // summed duration of the tiled event-kernel launches of the last iteration
        if (w->tk_used == 0) return -1;         // (one launch per batch of events; synchronises on the last one)
        double total = 0.0;
        for (size_t i = 0; i + 1 < w->tk_used; i += 2) {
            float ms = 0.f;
            if (cudaEventSynchronize(w->tk[i + 1]) != cudaSuccess || cudaEventElapsedTime(&ms, w->tk[i], w->tk[i + 1]) != cudaSuccess) return -1;
            total += ms;
        }
        return (int64_t)(total * 1e6);
    }
    if (!strcmp(name, "last_kernel_launches")) return (int64_t)(w->tk_used / 2);
    if (!strcmp(name, "last_variant")) return w->plan.shape;
    if (!strcmp(name, "last_variant_low")) return w->plan.dp.n_cls == 2 ? w->plan.shape_lo : -1;
    if (!strcmp(name, "last_smem_bytes")) return (int64_t)w->plan.smem;
    if (!strcmp(name, "last_tiled")) return w->plan.dp.t_max >= 0.f;
    if (!strcmp(name, "last_overflow")) {       // records the event kernel could not hold (0 by construction; synchronises the device)
        unsigned long long h = 0;
        if (!w->counters || cudaMemcpy(&h, w->counters + 2, sizeof h, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
        return (int64_t)h;
    }
    return -1;
}

uint64_t jpet_launch_count(void) { return g_launches.load(); }

void jpet_release(void) {
    int cur = -1;
    cudaGetDevice(&cur);
    for (auto& kv : g_ctx) {
        if (cudaSetDevice(kv.first) == cudaSuccess) release_ws(*kv.second);
    }
    g_ctx.clear();
    if (cur >= 0) cudaSetDevice(cur);
}

const char* jpet_last_error(void) { return g_err.c_str(); }

int64_t jpet_plan_describe(const jpet_geometry* geometry, const jpet_sigmas* sigmas, const jpet_grid* grid, int64_t* out,
                           int32_t n_out, uint32_t* task_table_host, int64_t table_cap) {
    g_err.clear();
    int rc = validate(geometry, sigmas, grid);
    if (rc) return rc;
    if (!sigmas) return fail(JPET_E_INVAL, "NULL sigmas");
    if (!out || n_out < 17) return fail(JPET_E_INVAL, "out must hold at least 17 values");
    jpet_host::RowsPlan plan;
    std::vector<uint32_t> tab;
    make_plan(*geometry, *sigmas, *grid, &plan, &tab);
    const DevParams& dp = plan.dp;
    const bool tiled = dp.t_max >= 0.f;
    const Shape v = tiled ? kShapes[plan.shape] : Shape{"none", 0, 0, 0, 0, 0, 0, 0, 0, 0};
    const int64_t vals[17] = {plan.shape, v.DEG, v.NWE, v.NG, v.NJA, v.NJB, dp.HS, dp.WZ, dp.Sy, dp.Sz, dp.Hy, dp.Hz, dp.chunk,
                              (int64_t)plan.smem, tiled, dp.nr_min, dp.nr_max};
    for (int i = 0; i < 17; ++i) out[i] = vals[i];
    if (n_out >= 18) out[17] = tiled ? plan.shape_lo : -1;
    if (task_table_host)
        for (int64_t i = 0; i < std::min<int64_t>(table_cap, (int64_t)tab.size()); ++i) task_table_host[i] = tab[(size_t)i];
    return (int64_t)tab.size();
}

const char* jpet_shape_name(int32_t shape) { return shape >= 0 && shape < kNumShapes ? kShapes[shape].name : ""; }

int jpet_mlem_iterate_noalloc(const float* events_dev, int64_t n, const jpet_geometry* geometry, const jpet_sigmas* sigmas,
                              const jpet_grid* grid, const float* rho_in_dev, float* rho_out_dev, void* cuda_stream) {
    g_err.clear();
    int rc = validate(geometry, sigmas, grid);
    if (rc) return rc;
    if (!sigmas) return fail(JPET_E_INVAL, "NULL sigmas");
    if (n < 0 || (n > 0 && !events_dev)) return fail(JPET_E_INVAL, "bad events");
    if (n > 0x7fffffffll) return fail(JPET_E_INVAL, "jpet_mlem_iterate_noalloc takes at most 2^31 - 1 events per call");
    if (!rho_in_dev || !rho_out_dev) return fail(JPET_E_INVAL, "NULL image pointer");
    const int64_t M64 = (int64_t)grid->n_y * grid->n_z;
    if (M64 > kNoAllocMaxPixels)
        return fail(JPET_E_INVAL, "jpet_mlem_iterate_noalloc: an image of %d x %d = %lld pixels does not fit the static scratch "
                    "(JPET_NOALLOC_MAX_PIXELS = %d); use jpet_mlem_iterate, which allocates its workspace", grid->n_y, grid->n_z,
                    (long long)M64, kNoAllocMaxPixels);
    NoAllocDevice d;
    if ((rc = noalloc_device(&d))) return rc;        // first call on this device: cudaGetSymbolAddress + one attribute query
    const int M = (int)M64;
    float* s = reinterpret_cast<float*>(d.base);
    float* wT = reinterpret_cast<float*>(d.base + kNoAllocImageBytes);
    float* accT = reinterpret_cast<float*>(d.base + 2 * kNoAllocImageBytes);
    unsigned long long* counters = reinterpret_cast<unsigned long long*>(d.base + kNoAllocCountersAt);
    int* meta = reinterpret_cast<int*>(d.base + kNoAllocMetaAt);
    jpet_host::RowsPlan plan;
    make_plan(*geometry, *sigmas, *grid, &plan);     // host arithmetic only: the constants of Eq. 7-12 in plan.dp
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // the array keeps what the previous call left: s and w are rewritten in full for this grid, the accumulator and the
    // counters are zeroed by the pre-pass, the meta words are rewritten
    jpet::sensitivity_kernel<<<grid_for(M), 256, 0, st>>>(s, grid->n_y, grid->n_z, grid->pixel, geometry->R, geometry->L);
    jpet::prepass_kernel<<<grid_for(M), 256, 0, st>>>(s, rho_in_dev, wT, accT, grid->n_y, grid->n_z, counters);
    noalloc_meta_kernel<<<1, 32, 0, st>>>(meta, (int)n);
    jpet::mlem_rows_direct_kernel<false><<<d.sm_count * 16, 128, 0, st>>>(events_dev, 3, meta, plan.dp, wT, accT, counters, 0);
    jpet::PeerAcc pa{};
    pa.acc[0] = accT;
    pa.n = 1;
    jpet::finalise_kernel<<<grid_for(M), 256, 0, st>>>(s, rho_in_dev, pa, rho_out_dev, grid->n_y, grid->n_z);
    g_launches += 5;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

int jpet_abi_version(void) { return JPET_ABI_VERSION; }

}  // extern "C"
