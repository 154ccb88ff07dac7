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
#include <vector>

#include "mlem_kernels.cuh"
#include "mlem_rows2.cuh"
#include "mlem_rows3.cuh"
#include "task_table.h"

namespace {

using jpet::DevParams;

thread_local std::string g_err;
std::atomic<uint64_t> g_launches{0};
float g_a3_coef = 2.0f;
float g_gamma = 0.0f;             // off-diagonal coefficient of C^-1 (Eq. 12); 0 = the paper's diagonal case
int64_t g_opt_force_direct = 0;  // 1 = every event takes the direct (global-memory) path
int64_t g_opt_chunk = 0;         // events per work item, 0 = automatic
int64_t g_opt_sz = 0;            // sub-tile width in pixels, 0 = automatic
int64_t g_opt_time_kernel = 0;   // 1 = bracket the tiled event kernel with CUDA events (bench.py's roofline)
std::vector<cudaEvent_t> g_tk;    // event pairs around the tiled event kernel launches since the last begin
size_t g_tk_used = 0;
int64_t g_opt_variant = -1;      // -1 = automatic
int64_t g_opt_pdl = 1;           // 1 = launch the kernels of an iteration with programmatic stream serialisation
int64_t g_opt_poly_off = 0;      // 1 = never pick a polynomial-exponent variant automatically
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

// One batch of events sorted by sub-tile, with its work-item list (device memory).
struct BinSet {
    float* sorted = nullptr;            // [n][stride], regular bins first, the direct bin last
    int stride = 3;                     // floats per event: 3 = raw triple, 16 = EventRec (second-generation kernel)
    jpet::WorkItem* items = nullptr;
    int* meta = nullptr;                // 0: #items, 1: direct start, 2: direct count, 3: work counter
    int64_t n = 0;
    size_t cap_events = 0, cap_items = 0;
    bool owns_sorted = true;
};

struct PlanKey {
    jpet_geometry g; jpet_sigmas sg; jpet_grid gr; float a3, gamma;
    int64_t variant, sz, chunk, force_direct;
};

struct Workspace {
    // problem the workspace is currently set up for
    jpet_geometry geom{0, 0};
    jpet_sigmas sig{0, 0};
    jpet_grid grid{0, 0, 0};
    bool s_valid = false;
    bool open = false;          // between begin and end
    int M = 0;
    DevParams dp{};
    int variant = 0;
    size_t smem = 0;
    // device buffers
    float* s = nullptr;
    float* wT = nullptr;
    float* accT = nullptr;
    float* rho_a = nullptr;
    float* rho_b = nullptr;
    unsigned long long* counters = nullptr;
    size_t cap_M = 0;
    int* bin_of = nullptr;      // scratch of the binning pass
    size_t cap_bin_of = 0;
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
    PlanKey plan_key{};
    bool plan_valid = false;
    uint32_t* tab = nullptr;    // task table of the third-generation kernel (device copy of tab_host)
    size_t cap_tab = 0;
    std::vector<uint32_t> tab_host, tab_uploaded;
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
        // Eq. 12 is positive definite for gamma^2 < 1 / (2 sigma_z^2 sigma_dl^2); half of that keeps D > 0 as well
        // (a.C^-1.a changes by at most 2 |gamma| k y sigma_z^2 sin(theta) / R of itself)
        if (std::fabs((double)g_gamma) * std::sqrt(2.0) * sg->sigma_z * sg->sigma_dl > 0.5)
            return fail(JPET_E_INVAL, "|gamma| must be at most 0.5 / (sqrt(2) sigma_z sigma_dl) (Eq. 12 positive definite, D > 0)");
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

int ensure_images(int M) {
    if ((size_t)M > g_ws.cap_M) {
        cudaFree(g_ws.s); cudaFree(g_ws.wT); cudaFree(g_ws.accT); cudaFree(g_ws.rho_a); cudaFree(g_ws.rho_b);
        g_ws.s = g_ws.wT = g_ws.accT = g_ws.rho_a = g_ws.rho_b = nullptr;
        g_ws.cap_M = 0;
        CUDA_TRY(cudaMalloc(&g_ws.s, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&g_ws.wT, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&g_ws.accT, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&g_ws.rho_a, sizeof(float) * M));
        CUDA_TRY(cudaMalloc(&g_ws.rho_b, sizeof(float) * M));
        g_ws.cap_M = M;
        g_ws.s_valid = false;
    }
    if (!g_ws.counters) CUDA_TRY(cudaMalloc(&g_ws.counters, 4 * sizeof(unsigned long long)));
    return JPET_OK;
}

// ---- event-kernel variants: NW warps per CTA, rows split in NH parts, NR row passes, NJ cached pixels,
// HS = region row stride (compile time, so every shared-memory access has an immediate offset) ---------------
// Second-generation shapes (mlem_rows2.cuh) have NA > 0: NA blocks of 32 central rows, NH parts per row, NBW = 1
// adds the warp that takes the cap rows; NW = NA * NH + NBW.
struct Variant { int NW, NH, NR, NJ, HS, U, CF, MINB, PK, NA, NBW; };
constexpr Variant kVariants[] = {
    {1, 1, 1, 12, 64, 4, 1, 1, 0},    // 0: <= 32 rows, chords <= 12 px                            (config 1)
    {2, 1, 1, 20, 64, 4, 1, 10, 0},   // 1: <= 64 rows, chords <= 20 px, <= 96 registers           (configs 2, 3)
    {4, 2, 1, 12, 64, 4, 1, 1, 0},    // 2: <= 64 rows, chords <= 24 px in two halves
    {4, 1, 1, 36, 128, 4, 1, 1, 0},   // 3: <= 128 rows, chords <= 36 px
    {8, 2, 1, 20, 128, 4, 1, 1, 0},   // 4: <= 128 rows, chords <= 40 px in two halves             (config 4)
    {8, 2, 1, 24, 160, 4, 1, 1, 0},   // 5: <= 128 rows, chords <= 48 px in two halves
    {4, 1, 1, 44, 160, 4, 1, 1, 0},   // 6: <= 128 rows, chords <= 44 px                           (config 5)
    {1, 1, 2, 20, 64, 4, 1, 1, 0},    // 7: <= 64 rows in two passes of one warp, chords <= 20 px
    {2, 1, 1, 20, 64, 4, 1, 10, 1},   // 8: as 1, packed fp32x2 arithmetic
    {8, 2, 1, 20, 128, 4, 1, 1, 1},   // 9: as 4, packed
    {4, 1, 1, 44, 160, 4, 1, 1, 1},   // 10: as 6, packed
    {1, 1, 1, 12, 64, 4, 1, 1, 1},    // 11: as 0, packed
    {2, 1, 1, 20, 64, 4, 1, 10, 1, 1, 1},    // 12: rows2, 32 central rows + cap warp, chords <= 20      (configs 2, 3)
    {2, 1, 1, 20, 64, 4, 1, 10, 0, 1, 1},    // 13: as 12, scalar arithmetic
    {1, 1, 1, 12, 64, 4, 1, 1, 1, 1, 0},     // 14: rows2, <= 32 rows, chords <= 12                       (config 1)
    {7, 2, 1, 20, 128, 4, 1, 1, 1, 3, 1},    // 15: rows2, 96 central rows in halves + cap warp, chords <= 40 (config 4)
    {8, 2, 1, 24, 160, 4, 1, 1, 1, 4, 0},    // 16: rows2, <= 128 rows in halves, chords <= 48            (config 5)
    {8, 2, 1, 20, 128, 4, 1, 1, 1, 4, 0},    // 17: rows2, <= 128 rows in halves, chords <= 40
    {7, 2, 1, 24, 160, 4, 1, 1, 1, 3, 1},    // 18: rows2, 96 central rows in halves + cap warp, chords <= 48
    {4, 1, 1, 44, 160, 4, 1, 1, 1, 4, 0},    // 19: rows2, <= 128 rows, chords <= 44
    {4, 1, 1, 36, 128, 4, 1, 1, 1, 3, 1},    // 20: rows2, 96 central rows + cap warp, chords <= 36
};
constexpr int kNumVariants2 = sizeof(kVariants) / sizeof(kVariants[0]);
// Third-generation shapes (mlem_rows3.cuh), variant id = kNumVariants2 + index: NWE warps per event, NG event groups
// per CTA, NJA / NJB pixel capacity of the two pieces a lane walks (NJB = 0: one piece), region row stride HS.
// DEG: 0 = closed form (rsqrt + ex2 per pixel), 4 / 5 = exponent as a polynomial in u (one ex2 per pixel; make_plan
// bounds the truncation error and picks the degree); BW: pixels per block of the walks.
struct Variant3 { int NWE, NG, NJA, NJB, HS, MINB, DEG, BW; };
constexpr Variant3 kVariants3[] = {
    {1, 4, 20, 8, 64, 4, 0, 8},      // 21: <= 64 rows, chords <= 20 px, four independent warps per CTA      (configs 2, 3)
    {1, 4, 12, 0, 64, 4, 0, 8},      // 22: <= 32 rows, chords <= 12 px                                     (config 1)
    {4, 1, 36, 0, 128, 1, 0, 8},     // 23: <= 128 rows, chords <= 36 px, one row per lane                   (config 4)
    {4, 1, 44, 0, 128, 1, 0, 8},     // 24: <= 128 rows, chords <= 44 px, one row per lane                   (config 5)
    {2, 2, 36, 28, 128, 1, 0, 8},    // 25: <= 128 rows on two warps: 64 central rows + caps, chords <= 36
    {1, 8, 20, 8, 64, 2, 0, 8},      // 26: as 21, eight warps per CTA
    {1, 2, 20, 8, 64, 8, 0, 8},      // 27: as 21, two warps per CTA
    {1, 4, 20, 8, 64, 3, 0, 8},      // 28: as 21, at most 3 CTAs per SM (more registers)
    {1, 4, 20, 8, 64, 2, 0, 8},      // 29: as 21, at most 2 CTAs per SM
    {1, 4, 20, 8, 64, 4, 4, 4},      // 30: as 21, polynomial exponent of degree 4, blocks of 4          (configs 2, 3)
    {1, 4, 12, 0, 64, 4, 4, 4},      // 31: as 22, degree 4                                              (config 1)
    {4, 1, 36, 0, 128, 1, 5, 8},     // 32: as 23, degree 5                                              (config 4)
    {4, 1, 44, 0, 128, 1, 4, 8},     // 33: as 24, degree 4                                              (config 5)
    {1, 4, 20, 8, 64, 4, 5, 4},      // 34: as 30, degree 5
    {1, 4, 12, 0, 64, 4, 5, 4},      // 35: as 31, degree 5
    {4, 1, 36, 0, 128, 1, 4, 8},     // 36: as 32, degree 4
    {4, 1, 44, 0, 128, 1, 5, 8},     // 37: as 33, degree 5
    {1, 4, 20, 8, 64, 4, 4, 8},      // 38: as 30, blocks of 8
    {1, 4, 20, 8, 64, 4, 0, 4},      // 39: as 21, blocks of 4
    {1, 4, 12, 0, 64, 4, 4, 8},      // 40: as 31, blocks of 8
    {1, 4, 12, 0, 64, 4, 5, 8},      // 41: as 40, degree 5
    {1, 4, 20, 8, 64, 4, 5, 8},      // 42: as 38, degree 5
    {4, 4, 36, 0, 128, 1, 5, 8},     // 43: as 32, four event groups per CTA (one CTA of 16 warps per SM)
    {4, 4, 44, 0, 128, 1, 4, 8},     // 44: as 33, four event groups per CTA
    {4, 3, 36, 0, 128, 1, 5, 8},     // 45: as 32, three event groups per CTA
    {4, 3, 44, 0, 128, 1, 4, 8},     // 46: as 33, three event groups per CTA
    {4, 4, 36, 0, 128, 1, 0, 8},     // 47: as 43, closed form
    {4, 4, 44, 0, 128, 1, 0, 8},     // 48: as 44, closed form
    {4, 4, 36, 0, 128, 1, 4, 8},     // 49: as 43, degree 4
    {4, 4, 44, 0, 128, 1, 5, 8},     // 50: as 44, degree 5
    {1, 4, 20, 8, 64, 4, 4, 16},     // 51: as 38, blocks of 16 (config 2: 0.728 -> 0.710 ms)             (configs 2, 3)
    {4, 4, 44, 0, 128, 1, 4, 16},    // 52: as 44, blocks of 16                                          (config 5)
    {4, 4, 36, 0, 128, 1, 5, 16},    // 53: as 43, blocks of 16                                          (config 4)
    {3, 4, 36, 8, 128, 1, 5, 16},    // 54: three warps per event: 96 central rows + the few rows beyond them as B pieces (config 4)
    {3, 4, 44, 8, 128, 1, 4, 16},    // 55: as 54 for chords of up to 44 pixels, degree 4
    {1, 4, 20, 8, 64, 4, 4, 32},     // 56: as 51, one block per piece (config 2: 0.694 -> 0.680 ms)       (configs 2, 3)
    {4, 4, 44, 0, 128, 1, 4, 32},    // 57: as 52, blocks of 32
    {3, 4, 36, 8, 128, 1, 5, 32},    // 58: as 54, blocks of 32 (13.96 -> 13.08 ms per 5x10^6 events)       (config 4)
    {1, 4, 12, 0, 64, 4, 4, 16},     // 59: as 40, one block per piece
    {1, 4, 12, 0, 64, 4, 0, 16},     // 60: as 22 (closed form), one block per piece (fig4: 0.813 -> 0.794 ms)   (fig4)
};
// shapes in order of size: closed-form / degree-4 / degree-5 instances of each
constexpr int kShape3[4][3] = {{39, 19, 20}, {0, 35, 21}, {26, 28, 32}, {27, 31, 29}};
constexpr int kNumVariants3 = sizeof(kVariants3) / sizeof(kVariants3[0]);
constexpr int kNumVariants = kNumVariants2 + kNumVariants3;

int batch_chunk(int64_t n, const DevParams& dp);

// Kernel launch with the programmatic-stream-serialisation attribute (PDL): the kernel may be scheduled while the
// previous kernel of the stream drains; every kernel launched this way starts with pdl_wait() (mlem_kernels.cuh), so
// it reads nothing the previous kernel wrote before that kernel has completed.  Hides most of the launch gaps between
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
    cfg.numAttrs = g_opt_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

template <int NW, int NH, int NR, int NJ, int HS, int U, bool CF, int MINB, bool PK>
int launch_rows(const BinSet& bs, const DevParams& dp, size_t smem, cudaStream_t stream) {
    auto kern = jpet::mlem_rows_kernel<NW, NH, NR, NJ, HS, U, CF, MINB, PK>;
    if (bs.stride != 3) return fail(JPET_E_INVAL, "internal: first-generation kernel needs raw event triples");
    if (dp.t_max >= 0.f) {     // tiled path
        if (dp.HS != HS) return fail(JPET_E_INVAL, "internal: region stride %d does not match the kernel's %d", dp.HS, HS);
        static size_t attr_set = 0;
        if (smem > 40 * 1024 && smem > attr_set) {
            CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            attr_set = smem;
        }
        int per_sm = 0;
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NW * 32, smem));
        if (per_sm < 1) return fail(JPET_E_CUDA, "event kernel does not fit on an SM (%zu B of shared memory)", smem);
        if (g_opt_ctas_per_sm > 0) per_sm = (int)std::min<int64_t>(per_sm, g_opt_ctas_per_sm);
        int64_t max_items = bs.n / batch_chunk(bs.n, dp) + (int64_t)dp.nby * dp.nbz + 1;
        int grid = (int)std::min<int64_t>((int64_t)g_ws.sm_count * per_sm, std::max<int64_t>(max_items, 1));
        if (g_opt_time_kernel) {
            if (g_tk_used + 2 > g_tk.size()) {
                g_tk.resize(g_tk_used + 2, nullptr);
                CUDA_TRY(cudaEventCreate(&g_tk[g_tk_used])); CUDA_TRY(cudaEventCreate(&g_tk[g_tk_used + 1]));
            }
            CUDA_TRY(cudaEventRecord(g_tk[g_tk_used], stream));
        }
        kern<<<grid, NW * 32, smem, stream>>>(bs.sorted, bs.items, bs.meta, dp, g_ws.wT, g_ws.accT, g_ws.counters);
        g_launches++;
        if (g_opt_time_kernel) { CUDA_TRY(cudaEventRecord(g_tk[g_tk_used + 1], stream)); g_tk_used += 2; }
        CUDA_TRY(cudaGetLastError());
    }
    // direct path for the events of the last bin (all events when no region fits shared memory)
    int dgrid = dp.t_max >= 0.f ? g_ws.sm_count : g_ws.sm_count * 16;
    CUDA_TRY(launch_pdl(jpet::mlem_rows_direct_kernel, dim3(dgrid), dim3(128), 0, stream, bs.sorted, bs.stride, bs.meta, dp, g_ws.wT,
                        g_ws.accT, g_ws.counters));
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

template <int NA, int NH, int NBW, int NJ, int HS, int U, bool PK, int MINB>
int launch_rows2(const BinSet& bs, const DevParams& dp, size_t smem, cudaStream_t stream) {
    constexpr int NW = NA * NH + NBW;
    auto kern = jpet::mlem_rows2_kernel<NA, NH, NBW, NJ, HS, U, PK, MINB>;
    if (bs.stride != 16) return fail(JPET_E_INVAL, "internal: rows2 kernel needs event records");
    if (dp.t_max >= 0.f) {
        if (dp.HS != HS) return fail(JPET_E_INVAL, "internal: region stride %d does not match the kernel's %d", dp.HS, HS);
        static size_t attr_set = 0;
        if (smem > 40 * 1024 && smem > attr_set) {
            CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            attr_set = smem;
        }
        int per_sm = 0;
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NW * 32, smem));
        if (per_sm < 1) return fail(JPET_E_CUDA, "event kernel does not fit on an SM (%zu B of shared memory)", smem);
        if (g_opt_ctas_per_sm > 0) per_sm = (int)std::min<int64_t>(per_sm, g_opt_ctas_per_sm);
        int64_t max_items = bs.n / batch_chunk(bs.n, dp) + (int64_t)dp.nby * dp.nbz + 1;
        int grid = (int)std::min<int64_t>((int64_t)g_ws.sm_count * per_sm, std::max<int64_t>(max_items, 1));
        if (g_opt_time_kernel) {
            if (g_tk_used + 2 > g_tk.size()) {
                g_tk.resize(g_tk_used + 2, nullptr);
                CUDA_TRY(cudaEventCreate(&g_tk[g_tk_used])); CUDA_TRY(cudaEventCreate(&g_tk[g_tk_used + 1]));
            }
            CUDA_TRY(cudaEventRecord(g_tk[g_tk_used], stream));
        }
        kern<<<grid, NW * 32, smem, stream>>>(reinterpret_cast<const jpet::EventRec*>(bs.sorted), bs.items, bs.meta, dp,
                                             g_ws.wT, g_ws.accT, g_ws.counters);
        g_launches++;
        if (g_opt_time_kernel) { CUDA_TRY(cudaEventRecord(g_tk[g_tk_used + 1], stream)); g_tk_used += 2; }
        CUDA_TRY(cudaGetLastError());
    }
    int dgrid = dp.t_max >= 0.f ? g_ws.sm_count : g_ws.sm_count * 16;
    CUDA_TRY(launch_pdl(jpet::mlem_rows_direct_kernel, dim3(dgrid), dim3(128), 0, stream, bs.sorted, bs.stride, bs.meta, dp, g_ws.wT,
                        g_ws.accT, g_ws.counters));
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

template <int NWE, int NG, int NJA, int NJB, int HS, int MINB, int DEG, int BW>
int launch_rows3(const BinSet& bs, const DevParams& dp, size_t smem, cudaStream_t stream) {
    constexpr int NT = NWE * NG * 32;
    auto kern = jpet::mlem_rows3_kernel<NWE, NG, NJA, NJB, HS, MINB, DEG, BW>;
    if (bs.stride != 16) return fail(JPET_E_INVAL, "internal: rows3 kernel needs event records");
    if (dp.t_max >= 0.f) {
        if (dp.HS != HS) return fail(JPET_E_INVAL, "internal: region stride %d does not match the kernel's %d", dp.HS, HS);
        static size_t attr_set = 0;
        if (smem > 40 * 1024 && smem > attr_set) {
            CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            attr_set = smem;
        }
        int per_sm = 0;
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
        if (per_sm < 1) return fail(JPET_E_CUDA, "event kernel does not fit on an SM (%zu B of shared memory)", smem);
        if (g_opt_ctas_per_sm > 0) per_sm = (int)std::min<int64_t>(per_sm, g_opt_ctas_per_sm);
        int64_t max_items = bs.n / batch_chunk(bs.n, dp) + (int64_t)dp.nby * dp.nbz + 1;
        int grid = (int)std::min<int64_t>((int64_t)g_ws.sm_count * per_sm, std::max<int64_t>(max_items, 1));
        if (g_opt_time_kernel) {
            if (g_tk_used + 2 > g_tk.size()) {
                g_tk.resize(g_tk_used + 2, nullptr);
                CUDA_TRY(cudaEventCreate(&g_tk[g_tk_used])); CUDA_TRY(cudaEventCreate(&g_tk[g_tk_used + 1]));
            }
            CUDA_TRY(cudaEventRecord(g_tk[g_tk_used], stream));
        }
        CUDA_TRY(launch_pdl(kern, dim3(grid), dim3(NT), smem, stream, reinterpret_cast<const jpet::EventRec*>(bs.sorted), bs.items,
                            bs.meta, dp, g_ws.wT, g_ws.accT, g_ws.tab, g_ws.counters));
        g_launches++;
        if (g_opt_time_kernel) { CUDA_TRY(cudaEventRecord(g_tk[g_tk_used + 1], stream)); g_tk_used += 2; }
        CUDA_TRY(cudaGetLastError());
    }
    int dgrid = dp.t_max >= 0.f ? g_ws.sm_count : g_ws.sm_count * 16;
    CUDA_TRY(launch_pdl(jpet::mlem_rows_direct_kernel, dim3(dgrid), dim3(128), 0, stream, bs.sorted, bs.stride, bs.meta, dp, g_ws.wT,
                        g_ws.accT, g_ws.counters));
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

int dispatch_rows(int variant, const BinSet& bs, const DevParams& dp, size_t smem, cudaStream_t st) {
    switch (variant) {
        case kNumVariants2 + 0: return launch_rows3<1, 4, 20, 8, 64, 4, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 1: return launch_rows3<1, 4, 12, 0, 64, 4, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 2: return launch_rows3<4, 1, 36, 0, 128, 1, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 3: return launch_rows3<4, 1, 44, 0, 128, 1, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 4: return launch_rows3<2, 2, 36, 28, 128, 1, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 5: return launch_rows3<1, 8, 20, 8, 64, 2, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 6: return launch_rows3<1, 2, 20, 8, 64, 8, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 7: return launch_rows3<1, 4, 20, 8, 64, 3, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 8: return launch_rows3<1, 4, 20, 8, 64, 2, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 9: return launch_rows3<1, 4, 20, 8, 64, 4, 4, 4>(bs, dp, smem, st);
        case kNumVariants2 + 10: return launch_rows3<1, 4, 12, 0, 64, 4, 4, 4>(bs, dp, smem, st);
        case kNumVariants2 + 11: return launch_rows3<4, 1, 36, 0, 128, 1, 5, 8>(bs, dp, smem, st);
        case kNumVariants2 + 12: return launch_rows3<4, 1, 44, 0, 128, 1, 4, 8>(bs, dp, smem, st);
        case kNumVariants2 + 13: return launch_rows3<1, 4, 20, 8, 64, 4, 5, 4>(bs, dp, smem, st);
        case kNumVariants2 + 14: return launch_rows3<1, 4, 12, 0, 64, 4, 5, 4>(bs, dp, smem, st);
        case kNumVariants2 + 15: return launch_rows3<4, 1, 36, 0, 128, 1, 4, 8>(bs, dp, smem, st);
        case kNumVariants2 + 16: return launch_rows3<4, 1, 44, 0, 128, 1, 5, 8>(bs, dp, smem, st);
        case kNumVariants2 + 17: return launch_rows3<1, 4, 20, 8, 64, 4, 4, 8>(bs, dp, smem, st);
        case kNumVariants2 + 18: return launch_rows3<1, 4, 20, 8, 64, 4, 0, 4>(bs, dp, smem, st);
        case kNumVariants2 + 19: return launch_rows3<1, 4, 12, 0, 64, 4, 4, 8>(bs, dp, smem, st);
        case kNumVariants2 + 20: return launch_rows3<1, 4, 12, 0, 64, 4, 5, 8>(bs, dp, smem, st);
        case kNumVariants2 + 21: return launch_rows3<1, 4, 20, 8, 64, 4, 5, 8>(bs, dp, smem, st);
        case kNumVariants2 + 22: return launch_rows3<4, 4, 36, 0, 128, 1, 5, 8>(bs, dp, smem, st);
        case kNumVariants2 + 23: return launch_rows3<4, 4, 44, 0, 128, 1, 4, 8>(bs, dp, smem, st);
        case kNumVariants2 + 24: return launch_rows3<4, 3, 36, 0, 128, 1, 5, 8>(bs, dp, smem, st);
        case kNumVariants2 + 25: return launch_rows3<4, 3, 44, 0, 128, 1, 4, 8>(bs, dp, smem, st);
        case kNumVariants2 + 26: return launch_rows3<4, 4, 36, 0, 128, 1, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 27: return launch_rows3<4, 4, 44, 0, 128, 1, 0, 8>(bs, dp, smem, st);
        case kNumVariants2 + 28: return launch_rows3<4, 4, 36, 0, 128, 1, 4, 8>(bs, dp, smem, st);
        case kNumVariants2 + 29: return launch_rows3<4, 4, 44, 0, 128, 1, 5, 8>(bs, dp, smem, st);
        case kNumVariants2 + 30: return launch_rows3<1, 4, 20, 8, 64, 4, 4, 16>(bs, dp, smem, st);
        case kNumVariants2 + 31: return launch_rows3<4, 4, 44, 0, 128, 1, 4, 16>(bs, dp, smem, st);
        case kNumVariants2 + 32: return launch_rows3<4, 4, 36, 0, 128, 1, 5, 16>(bs, dp, smem, st);
        case kNumVariants2 + 33: return launch_rows3<3, 4, 36, 8, 128, 1, 5, 16>(bs, dp, smem, st);
        case kNumVariants2 + 34: return launch_rows3<3, 4, 44, 8, 128, 1, 4, 16>(bs, dp, smem, st);
        case kNumVariants2 + 35: return launch_rows3<1, 4, 20, 8, 64, 4, 4, 32>(bs, dp, smem, st);
        case kNumVariants2 + 36: return launch_rows3<4, 4, 44, 0, 128, 1, 4, 32>(bs, dp, smem, st);
        case kNumVariants2 + 37: return launch_rows3<3, 4, 36, 8, 128, 1, 5, 32>(bs, dp, smem, st);
        case kNumVariants2 + 38: return launch_rows3<1, 4, 12, 0, 64, 4, 4, 16>(bs, dp, smem, st);
        case kNumVariants2 + 39: return launch_rows3<1, 4, 12, 0, 64, 4, 0, 16>(bs, dp, smem, st);
        case 0: return launch_rows<1, 1, 1, 12, 64, 4, true, 1, false>(bs, dp, smem, st);
        case 1: return launch_rows<2, 1, 1, 20, 64, 4, true, 10, false>(bs, dp, smem, st);
        case 2: return launch_rows<4, 2, 1, 12, 64, 4, true, 1, false>(bs, dp, smem, st);
        case 3: return launch_rows<4, 1, 1, 36, 128, 4, true, 1, false>(bs, dp, smem, st);
        case 4: return launch_rows<8, 2, 1, 20, 128, 4, true, 1, false>(bs, dp, smem, st);
        case 5: return launch_rows<8, 2, 1, 24, 160, 4, true, 1, false>(bs, dp, smem, st);
        case 6: return launch_rows<4, 1, 1, 44, 160, 4, true, 1, false>(bs, dp, smem, st);
        case 7: return launch_rows<1, 1, 2, 20, 64, 4, true, 1, false>(bs, dp, smem, st);
        case 8: return launch_rows<2, 1, 1, 20, 64, 4, true, 10, true>(bs, dp, smem, st);
        case 9: return launch_rows<8, 2, 1, 20, 128, 4, true, 1, true>(bs, dp, smem, st);
        case 10: return launch_rows<4, 1, 1, 44, 160, 4, true, 1, true>(bs, dp, smem, st);
        case 11: return launch_rows<1, 1, 1, 12, 64, 4, true, 1, true>(bs, dp, smem, st);
        case 12: return launch_rows2<1, 1, 1, 20, 64, 4, true, 10>(bs, dp, smem, st);
        case 13: return launch_rows2<1, 1, 1, 20, 64, 4, false, 10>(bs, dp, smem, st);
        case 14: return launch_rows2<1, 1, 0, 12, 64, 4, true, 1>(bs, dp, smem, st);
        case 15: return launch_rows2<3, 2, 1, 20, 128, 4, true, 1>(bs, dp, smem, st);
        case 16: return launch_rows2<4, 2, 0, 24, 160, 4, true, 1>(bs, dp, smem, st);
        case 17: return launch_rows2<4, 2, 0, 20, 128, 4, true, 1>(bs, dp, smem, st);
        case 18: return launch_rows2<3, 2, 1, 24, 160, 4, true, 1>(bs, dp, smem, st);
        case 19: return launch_rows2<4, 1, 0, 44, 160, 4, true, 1>(bs, dp, smem, st);
        case 20: return launch_rows2<3, 1, 1, 36, 128, 4, true, 1>(bs, dp, smem, st);
        default: return fail(JPET_E_INVAL, "unknown kernel variant %d", variant);
    }
}

// Constants of the event kernel (computed in double, rounded once), the tiling of the image into
// sub-tiles + halo regions, and the kernel variant.
void make_plan(const jpet_geometry& g, const jpet_sigmas& sg, const jpet_grid& gr, float a3, float gamma, DevParams* out,
               int* variant, size_t* smem_out, std::vector<uint32_t>* tab_out = nullptr) {
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
    // ellipse extents in pixels: half height 1.5 sigma_dl cos(theta), half width 3 sqrt(sz^2/2 + sdl^2 sin^2/4) (App. B)
    double t_max = ((double)g.L + 8.0 * sg.sigma_z) / (2.0 * g.R);
    double sin2 = t_max * t_max / (1.0 + t_max * t_max);
    double hy = 1.5 * sg.sigma_dl / px;
    double hz = 3.0 * std::sqrt(0.5 * (double)sg.sigma_z * sg.sigma_z + 0.25 * (double)sg.sigma_dl * sg.sigma_dl * sin2) / px;
    double chord = 6.0 * sg.sigma_z / std::sqrt(2.0) / px;
    int rows_max = std::min<int>(gr.n_y, (int)std::floor(2.0 * hy) + 2);
    int chord_max = std::min<int>(gr.n_z, (int)std::floor(chord) + 2);
    p.Hy = (int)std::ceil(hy) + 1;
    p.Hz = (int)std::ceil(hz) + 1;
    p.t_max = (float)t_max;
    // ellipse row counts a regular event can have (unclipped): hy_px * cos(theta) for |tan theta| <= t_max, +- rounding
    const int nr_hi = std::min(255, (int)std::floor(2.0 * hy) + 2);
    const int nr_lo = std::max(1, (int)std::floor(2.0 * hy / std::sqrt(1.0 + t_max * t_max)) - 1);
    // variant: smallest shape that holds rows_max rows, chord_max pixels per row, and the region's rows
    auto fits = [&](const Variant& c) {
        if (c.NA > 0) return rows_max + 1 <= 32 * (c.NA + c.NBW) && chord_max + 1 <= c.NJ * c.NH && 2 * p.Hy + 4 <= c.HS;
        return rows_max + 1 <= c.NW * 32 / c.NH * c.NR && chord_max <= c.NJ * c.NH && 2 * p.Hy + 4 <= c.HS;
    };
    std::vector<uint32_t> tab;
    auto fits3 = [&](const Variant3& c) {
        return 2 * p.Hy + 4 <= c.HS && jpet_host::build_task_table(nr_lo, nr_hi, (double)p.H0p, c.NWE, c.NJA, c.NJB, &tab);
    };
    int v = -1;
    if (g_opt_variant >= 0) v = (int)g_opt_variant;
    else {
        // third-generation shapes first; degree of the exponent polynomial from the truncation bound (mlem_rows3.cuh,
        // poly_coeffs2): |x| = |eps u / delta| <= xb, ba^2 / D <= eb inside the ellipse and the image
        const double y_max = 0.5 * gr.n_y * px, u_max = 3.0 * sg.sigma_z / std::sqrt(2.0), R2 = (double)g.R * g.R;
        // gamma (Eq. 12): delta changes by at most g_rel of itself, |b.C^-1.a| / sqrt(D) grows by at most g_ba
        const double ag = std::fabs((double)gamma);
        const double g_rel = 2.0 * ag * std::fabs((double)a3) * y_max * sg.sigma_z * sg.sigma_z * (t_max / std::sqrt(1.0 + t_max * t_max)) / g.R;
        const double g_ba = 6.0 / std::sqrt(2.0) * ag * sg.sigma_z * sg.sigma_dl;
        const double xb = 2.0 * (t_max / (1.0 + t_max * t_max)) * y_max * u_max / (R2 + y_max * y_max) / (0.95 - g_rel);
        const double eb = 1.1 * std::pow(3.0 * y_max / std::sqrt(R2 + y_max * y_max) + g_ba, 2.0);
        auto trunc_err = [&](int deg) {      // log2 units
            return 1.4427 * (0.5 * eb * std::pow(xb, deg - 1) / (1.0 - xb) + 0.5 * std::pow(xb, deg + 1) / (deg + 1));
        };
        const int deg_sel = g_opt_poly_off ? 0 : (trunc_err(4) <= 2e-5 ? 1 : (trunc_err(5) <= 2e-5 ? 2 : 0));
        // ellipses of at most ~100 rows on three warps instead of four (config 4: 91 rows on 128 lanes leave a quarter of
        // the lanes idle; 14.60 -> 14.02 ms per 5x10^6 events), the few rows beyond 96 as B pieces
        if (deg_sel == 2 && nr_hi > 64 && nr_hi <= 104 && fits3(kVariants3[37])) v = kNumVariants2 + 37;
        for (int sh = 0; sh < 4 && v < 0; ++sh)
            if (fits3(kVariants3[kShape3[sh][deg_sel]])) v = kNumVariants2 + kShape3[sh][deg_sel];
        const int order[] = {14, 12, 15, 16, 0, 8, 9, 10, 5};
        for (int cand : order)
            if (v < 0 && fits(kVariants[cand])) { v = cand; break; }
        if (v < 0) v = 5;
    }
    const bool gen3 = v >= kNumVariants2;
    // else: every event takes the direct path (the later generations have no overflow loops)
    bool tiles_ok;
    int v_HS, v_NJ, n_regions = 2;
    if (gen3) {
        const Variant3& c = kVariants3[v - kNumVariants2];
        tiles_ok = fits3(c);
        v_HS = c.HS; v_NJ = c.NJA; n_regions = 1 + c.NG;
        p.nr_min = nr_lo; p.nr_max = nr_hi;
    } else {
        tiles_ok = 2 * p.Hy + 4 <= kVariants[v].HS && (kVariants[v].NA == 0 || fits(kVariants[v]));
        v_HS = kVariants[v].HS; v_NJ = kVariants[v].NJ;
        p.nr_min = 0; p.nr_max = 0;
        tab.clear();
    }
    p.HS = v_HS;
    p.Sy = std::max(1, p.HS - 2 * p.Hy);
    // shared memory: w region + accumulator region(s) (+ task table).  The sub-tile width Sz (8 or 4 columns) is the
    // one that lets most warps live on an SM (228 KB per SM, 1 KB reserved per CTA, 227 KB per CTA); 8 on a tie.
    const size_t budget = 225 * 1024, sm_bytes = 228 * 1024, tab_bytes = tab.size() * sizeof(uint32_t);
    const int cta_warps = gen3 ? kVariants3[v - kNumVariants2].NWE * kVariants3[v - kNumVariants2].NG : kVariants[v].NW;
    size_t smem = 0;
    {
        int best_sz = 4;
        size_t best_warps = 0;
        for (int sz : {8, 4}) {
            if (g_opt_sz > 0) sz = (int)g_opt_sz;
            const size_t need = n_regions * sizeof(float) * (size_t)p.HS * (sz + 2 * p.Hz) + tab_bytes;
            const size_t ctas = need <= budget ? std::min<size_t>(sm_bytes / (need + 2048), 2048 / (32 * cta_warps)) : 0;
            if (ctas * cta_warps > best_warps) { best_warps = ctas * cta_warps; best_sz = sz; }
        }
        p.Sz = best_sz;
        p.WZ = p.Sz + 2 * p.Hz;
        smem = n_regions * sizeof(float) * (size_t)p.HS * p.WZ + tab_bytes;
    }
    if (smem > budget || !tiles_ok || p.WZ < v_NJ + 4 || g_opt_force_direct) { p.t_max = -1.f; smem = 0; p.nr_min = p.nr_max = 0; tab.clear(); }
    p.nby = (gr.n_y + 2 * p.Hy + p.Sy - 1) / p.Sy;
    p.nbz = (gr.n_z + 2 * p.Hz + p.Sz - 1) / p.Sz;
    // events per work item (one staging of w and one flush of the accumulator regions per item): measured optimum on B200
    // 128 events per group for the one-warp groups (config 2: 0.740 -> 0.734 ms), 256 for the four-warp groups
    // (configs 4, 5: +5-8 %)
    p.chunk = g_opt_chunk > 0 ? (int)g_opt_chunk
                              : (gen3 ? (kVariants3[v - kNumVariants2].NWE > 1 ? 256 : 128) * kVariants3[v - kNumVariants2].NG : 64);
    *out = p;
    *variant = v;
    *smem_out = smem;
    if (tab_out) tab_out->swap(tab);
}

bool same_problem(const jpet_geometry& g, const jpet_grid& gr) {
    return g_ws.s_valid && g_ws.geom.R == g.R && g_ws.geom.L == g.L && g_ws.grid.n_y == gr.n_y &&
           g_ws.grid.n_z == gr.n_z && g_ws.grid.pixel == gr.pixel;
}

int grid_for(int64_t M) { return (int)((M + 255) / 256); }

int plan_stride() { return (g_ws.variant >= kNumVariants2 || kVariants[g_ws.variant].NA > 0) ? 16 : 3; }

// Events per work item for a batch of n events: the plan's size, halved (not below 64) while the batch would give fewer
// than four items per SM - small batches are launch- and tail-bound.
int batch_chunk(int64_t n, const DevParams& dp) {
    int chunk = dp.chunk;
    if (g_opt_chunk > 0) return chunk;
    while (chunk > 64 && n / chunk < 4 * (int64_t)g_ws.sm_count) chunk /= 2;
    return chunk;
}

int ensure_binset(BinSet& bs, int64_t n, const DevParams& dp, bool need_sorted) {
    size_t items_cap = (size_t)(n / batch_chunk(n, dp)) + (size_t)dp.nby * dp.nbz + 2;
    bs.stride = plan_stride();
    const size_t need_floats = (size_t)bs.stride * (size_t)std::max<int64_t>(n, 1);
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
    if (!bs.meta) CUDA_TRY(cudaMalloc(&bs.meta, 4 * sizeof(int)));
    return JPET_OK;
}

void free_binset(BinSet& bs) {
    if (bs.owns_sorted) cudaFree(bs.sorted);
    cudaFree(bs.items);
    cudaFree(bs.meta);
    bs = BinSet{};
}

// Counting sort of one batch (<= kMaxBatch events) by sub-tile into bs.sorted, and its work items.
int bin_batch(const float* events, int64_t n, BinSet& bs, const DevParams& dp, cudaStream_t st) {
    const int nb = dp.nby * dp.nbz;
    if ((size_t)n > g_ws.cap_bin_of) {
        cudaFree(g_ws.bin_of);
        g_ws.bin_of = nullptr; g_ws.cap_bin_of = 0;
        CUDA_TRY(cudaMalloc(&g_ws.bin_of, sizeof(int) * (size_t)n));
        g_ws.cap_bin_of = (size_t)n;
    }
    if ((size_t)(2 * (nb + 1)) > g_ws.cap_counts) {
        cudaFree(g_ws.counts);
        g_ws.counts = nullptr; g_ws.cap_counts = 0;
        CUDA_TRY(cudaMalloc(&g_ws.counts, sizeof(int) * 2 * (size_t)(nb + 1)));
        g_ws.cap_counts = (size_t)(2 * (nb + 1));
        g_ws.counts_clean_nb = -1;
    }
    int* counts = g_ws.counts;
    int* cursors = g_ws.counts + (nb + 1);
    if (g_ws.counts_clean_nb != nb) {        // bin_scan_kernel leaves the counts zeroed: a memset only when the layout changes
        CUDA_TRY(cudaMemsetAsync(counts, 0, sizeof(int) * (nb + 1), st));
        g_ws.counts_clean_nb = nb;
    }
    const int per_block = jpet::kBinBlock * jpet::kBinPer;
    const int blocks = (int)((n + per_block - 1) / per_block);
    const int use_smem = nb + 1 <= jpet::kBinSmemMax;
    const size_t hist_bytes = use_smem ? sizeof(int) * (size_t)(nb + 1) : 0;
    if (n > 0) {
        CUDA_TRY(launch_pdl(jpet::bin_count_kernel, dim3(blocks), dim3(jpet::kBinBlock), hist_bytes, st, events, (int)n, dp, g_ws.bin_of,
                            counts, nb + 1, use_smem));
        g_launches++;
    }
    CUDA_TRY(launch_pdl(jpet::bin_scan_kernel, dim3(1), dim3(1024), 0, st, counts, cursors, bs.items, bs.meta, nb, batch_chunk(n, dp)));
    g_launches++;
    if (n > 0) {
        if (bs.stride == 16)
            CUDA_TRY(launch_pdl(jpet::bin_scatter_rec_kernel, dim3(blocks), dim3(jpet::kBinBlock), hist_bytes, st, events, (int)n,
                                g_ws.bin_of, cursors, reinterpret_cast<jpet::EventRec*>(bs.sorted), dp, nb + 1, use_smem));
        else
            jpet::bin_scatter_kernel<<<blocks, jpet::kBinBlock, hist_bytes, st>>>(events, (int)n, g_ws.bin_of, cursors, bs.sorted, nb + 1, use_smem);
        g_launches++;
    }
    CUDA_TRY(cudaGetLastError());
    bs.n = n;
    return JPET_OK;
}

int run_binset(BinSet& bs, cudaStream_t st) {
    // the work counter meta[3] is zero here: bin_scan_kernel zeroes it and mlem_rows_direct_kernel, the last kernel of every
    // run over a sorted set, zeroes it again
    return dispatch_rows(g_ws.variant, bs, g_ws.dp, g_ws.smem, st);
}

int do_begin(const jpet_geometry* g, const jpet_sigmas* sg, const jpet_grid* gr, const float* rho_in, cudaStream_t st) {
    int rc = validate(g, sg, gr);
    if (rc) return rc;
    if (!sg) return fail(JPET_E_INVAL, "NULL sigmas");
    if (!rho_in) return fail(JPET_E_INVAL, "NULL rho_in");
    if ((rc = ensure_device())) return rc;
    const int M = gr->n_y * gr->n_z;
    if ((rc = ensure_images(M))) return rc;
    if (!same_problem(*g, *gr)) {
        jpet::sensitivity_kernel<<<grid_for(M), 256, 0, st>>>(g_ws.s, gr->n_y, gr->n_z, gr->pixel, g->R, g->L);
        g_launches++;
        CUDA_TRY(cudaGetLastError());
        g_ws.geom = *g; g_ws.grid = *gr; g_ws.s_valid = true;
    }
    g_ws.sig = *sg; g_ws.M = M;
    {   // the plan depends only on these inputs: rebuild it (and the task table) when one of them changes
        const PlanKey key{*g, *sg, *gr, g_a3_coef, g_gamma, g_opt_variant, g_opt_sz, g_opt_chunk, g_opt_force_direct + 2 * g_opt_poly_off};
        if (!g_ws.plan_valid || memcmp(&key, &g_ws.plan_key, sizeof key) != 0) {
            make_plan(*g, *sg, *gr, g_a3_coef, g_gamma, &g_ws.dp, &g_ws.variant, &g_ws.smem, &g_ws.tab_host);
            g_ws.plan_key = key;
            g_ws.plan_valid = true;
        }
    }
    if (g_ws.variant < 0 || g_ws.variant >= kNumVariants) return fail(JPET_E_INVAL, "unknown kernel variant");
    if (!g_ws.tab_host.empty() && g_ws.tab_host != g_ws.tab_uploaded) {        // task table of the third-generation kernel
        if (g_ws.tab_host.size() > g_ws.cap_tab) {
            cudaFree(g_ws.tab);
            g_ws.tab = nullptr; g_ws.cap_tab = 0;
            CUDA_TRY(cudaMalloc(&g_ws.tab, sizeof(uint32_t) * g_ws.tab_host.size()));
            g_ws.cap_tab = g_ws.tab_host.size();
        }
        g_ws.tab_uploaded = g_ws.tab_host;      // the copy below reads tab_uploaded, which stays put until the next change
        CUDA_TRY(cudaMemcpyAsync(g_ws.tab, g_ws.tab_uploaded.data(), sizeof(uint32_t) * g_ws.tab_uploaded.size(),
                                 cudaMemcpyHostToDevice, st));
    }
    g_tk_used = 0;                 // last_kernel_ns covers the event-kernel launches of one iteration
    CUDA_TRY(launch_pdl(jpet::prepass_kernel, dim3(grid_for(M)), dim3(256), 0, st, (const float*)g_ws.s, rho_in, g_ws.wT, g_ws.accT,
                        gr->n_y, gr->n_z, g_ws.counters));
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
        int rc = ensure_binset(g_ws.scratch, nb, g_ws.dp, true);
        if (rc) return rc;
        if ((rc = bin_batch(events + 3 * off, nb, g_ws.scratch, g_ws.dp, st))) return rc;
        if ((rc = run_binset(g_ws.scratch, st))) return rc;
    }
    return JPET_OK;
}

int do_end(const float* rho_in, float* rho_out, cudaStream_t st) {
    if (!g_ws.open) return fail(JPET_E_INVAL, "jpet_mlem_end without jpet_mlem_begin");
    if (!rho_in || !rho_out) return fail(JPET_E_INVAL, "NULL image pointer");
    CUDA_TRY(launch_pdl(jpet::finalise_kernel, dim3(grid_for(g_ws.M)), dim3(256), 0, st, (const float*)g_ws.s, rho_in,
                        (const float*)g_ws.accT, rho_out, g_ws.grid.n_y, g_ws.grid.n_z));
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    g_ws.open = false;
    return JPET_OK;
}

// n_iter iterations over device-resident events; the events are binned once (first iteration) and the
// sorted copy is reused by the others (events never change between iterations).
int iterate_many(const float* events, int64_t n, const jpet_geometry* g, const jpet_sigmas* sg, const jpet_grid* gr,
                 const float* rho_start, float* rho_out, int n_iter, cudaStream_t st) {
    const int M = gr->n_y * gr->n_z;
    const float* cur = rho_start;
    const int64_t n_batches = (n + kMaxBatch - 1) / kMaxBatch;
    const bool keep = n_iter > 1;
    if (keep) while ((int64_t)g_ws.kept.size() < n_batches) g_ws.kept.emplace_back();
    for (int it = 0; it < n_iter; ++it) {
        float* nxt = (it == n_iter - 1) ? rho_out : (cur == g_ws.rho_a ? g_ws.rho_b : g_ws.rho_a);
        int rc = do_begin(g, sg, gr, cur, st);        // fixes the plan (kernel variant, record stride) for this problem
        if (rc) return rc;
        const size_t stride = (size_t)plan_stride();
        if (keep && it == 0 && stride * (size_t)n > g_ws.cap_kept_sorted) {      // capacity counts floats
            cudaFree(g_ws.kept_sorted);
            g_ws.kept_sorted = nullptr; g_ws.cap_kept_sorted = 0;
            CUDA_TRY(cudaMalloc(&g_ws.kept_sorted, sizeof(float) * stride * (size_t)n));
            g_ws.cap_kept_sorted = stride * (size_t)n;
        }
        if (!keep) {
            if ((rc = do_accumulate(events, n, st))) { g_ws.open = false; return rc; }
        } else {
            for (int64_t b = 0; b < n_batches; ++b) {
                BinSet& bs = g_ws.kept[b];
                int64_t off = b * kMaxBatch, nb = std::min(kMaxBatch, n - off);
                if (it == 0) {
                    bs.owns_sorted = false;
                    bs.sorted = g_ws.kept_sorted + stride * (size_t)off;
                    if ((rc = ensure_binset(bs, nb, g_ws.dp, false))) return rc;
                    if ((rc = bin_batch(events + 3 * off, nb, bs, g_ws.dp, st))) return rc;
                }
                if ((rc = run_binset(bs, st))) { g_ws.open = false; return rc; }
            }
        }
        if ((rc = do_end(cur, nxt, st))) return rc;
        cur = nxt;
    }
    (void)M;
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
    if ((rc = ensure_images(M))) return rc;
    // upload chunk: a quarter of the events, between 5x10^5 and 2x10^6, so that the copy of chunk c+1 overlaps the sort
    // and the event kernel of chunk c also for one-batch problems (config 2 on a box with a 12 GB/s host link:
    // 1.6 ms with one chunk, 1.07 ms with two; no difference on a 50 GB/s link)
    if (chunk <= 0) chunk = std::min<int64_t>(2000000, std::max<int64_t>(500000, (n + 3) / 4));
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
    if (n_iter > 0) {
        // first iteration: the upload of chunk c+1 overlaps the binning + event kernels of chunk c
        if ((rc = do_begin(g, sg, gr, cur, ks))) return rc;
        if ((rc = accumulate_from_host(events_host, n, chunk, fits, false))) return rc;
        if ((rc = do_end(cur, nxt, ks))) return rc;
        std::swap(cur, nxt);
        if (n_iter > 1) {
            if (fits) {         // events are now resident in the staging buffer: bin once, iterate
                if ((rc = iterate_many(g_ws.stage, n, g, sg, gr, cur, nxt, n_iter - 1, ks))) return rc;
                std::swap(cur, nxt);
            } else {
                for (int it = 1; it < n_iter; ++it) {
                    if ((rc = do_begin(g, sg, gr, cur, ks))) return rc;
                    if ((rc = accumulate_from_host(events_host, n, chunk, false, false))) return rc;
                    if ((rc = do_end(cur, nxt, ks))) return rc;
                    std::swap(cur, nxt);
                }
            }
        }
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
    if ((rc = ensure_images(M))) return rc;
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
    return iterate_many(events_dev, n, geometry, sigmas, grid, cur, rho_out_dev, n_iter, st);
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
    int variant = 0;
    size_t smem = 0;
    make_plan(*geometry, *sigmas, *grid, g_a3_coef, g_gamma, &dp, &variant, &smem);
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

int jpet_set_gamma(float gamma) {
    g_err.clear();
    if (!std::isfinite(gamma)) return fail(JPET_E_INVAL, "gamma must be finite");
    g_gamma = gamma;
    return JPET_OK;
}

float jpet_get_gamma(void) { return g_gamma; }

int jpet_set_option(const char* name, int64_t value) {
    g_err.clear();
    if (!name) return fail(JPET_E_INVAL, "NULL option name");
    if (!strcmp(name, "force_direct")) {
        if (value < 0 || value > 1) return fail(JPET_E_INVAL, "force_direct must be 0 or 1");
        g_opt_force_direct = value;
    } else if (!strcmp(name, "time_kernel")) {
        if (value < 0 || value > 1) return fail(JPET_E_INVAL, "time_kernel must be 0 or 1");
        g_opt_time_kernel = value;
        g_tk_used = 0;
    } else if (!strcmp(name, "sub_tile_z")) {
        if (value < 0 || value > 256) return fail(JPET_E_INVAL, "sub_tile_z must be 0 (auto) .. 256");
        g_opt_sz = value;
    } else if (!strcmp(name, "chunk")) {
        if (value < 0 || value > (1 << 20)) return fail(JPET_E_INVAL, "chunk must be 0 (auto) .. 2^20");
        g_opt_chunk = value;
    } else if (!strcmp(name, "variant")) {
        if (value < -1 || value >= kNumVariants) return fail(JPET_E_INVAL, "variant must be -1 (auto) .. %d", kNumVariants - 1);
        g_opt_variant = value;
    } else if (!strcmp(name, "poly_off")) {
        g_opt_poly_off = value != 0;
    } else if (!strcmp(name, "pdl")) {
        g_opt_pdl = value != 0;
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
    if (!strcmp(name, "force_direct")) return g_opt_force_direct;
    if (!strcmp(name, "chunk")) return g_opt_chunk;
    if (!strcmp(name, "sub_tile_z")) return g_opt_sz;
    if (!strcmp(name, "time_kernel")) return g_opt_time_kernel;
    if (!strcmp(name, "last_kernel_ns")) {      // summed duration of the tiled event-kernel launches of the last iteration
        if (g_tk_used == 0) return -1;          // (one launch per batch of events; synchronises on the last one)
        double total = 0.0;
        for (size_t i = 0; i + 1 < g_tk_used; i += 2) {
            float ms = 0.f;
            if (cudaEventSynchronize(g_tk[i + 1]) != cudaSuccess || cudaEventElapsedTime(&ms, g_tk[i], g_tk[i + 1]) != cudaSuccess) return -1;
            total += ms;
        }
        return (int64_t)(total * 1e6);
    }
    if (!strcmp(name, "last_kernel_launches")) return (int64_t)(g_tk_used / 2);
    if (!strcmp(name, "variant")) return g_opt_variant;
    if (!strcmp(name, "poly_off")) return g_opt_poly_off;
    if (!strcmp(name, "pdl")) return g_opt_pdl;
    if (!strcmp(name, "ctas_per_sm")) return g_opt_ctas_per_sm;
    if (!strcmp(name, "last_variant")) return g_ws.variant;
    if (!strcmp(name, "last_smem_bytes")) return (int64_t)g_ws.smem;
    if (!strcmp(name, "last_tiled")) return g_ws.dp.t_max >= 0.f;
    if (!strcmp(name, "last_overflow")) {       // pieces that exceeded their slot (0 by construction; synchronises the device)
        unsigned long long h = 0;
        if (!g_ws.counters || cudaMemcpy(&h, g_ws.counters + 2, sizeof h, cudaMemcpyDeviceToHost) != cudaSuccess) return -1;
        return (int64_t)h;
    }
    return -1;
}

uint64_t jpet_launch_count(void) { return g_launches.load(); }

void jpet_release(void) {
    cudaFree(g_ws.s); cudaFree(g_ws.wT); cudaFree(g_ws.accT); cudaFree(g_ws.rho_a); cudaFree(g_ws.rho_b);
    cudaFree(g_ws.counters); cudaFree(g_ws.stage); cudaFree(g_ws.bin_of); cudaFree(g_ws.counts); cudaFree(g_ws.kept_sorted);
    g_ws.counts_clean_nb = -1;
    cudaFree(g_ws.tab);
    free_binset(g_ws.scratch);
    for (auto& bs : g_ws.kept) free_binset(bs);
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

int64_t jpet_plan_describe(const jpet_geometry* geometry, const jpet_sigmas* sigmas, const jpet_grid* grid, int64_t* out,
                           int32_t n_out, uint32_t* task_table_host, int64_t table_cap) {
    g_err.clear();
    int rc = validate(geometry, sigmas, grid);
    if (rc) return rc;
    if (!sigmas) return fail(JPET_E_INVAL, "NULL sigmas");
    if (!out || n_out < 17) return fail(JPET_E_INVAL, "out must hold at least 17 values");
    DevParams dp;
    int variant = 0;
    size_t smem = 0;
    std::vector<uint32_t> tab;
    make_plan(*geometry, *sigmas, *grid, g_a3_coef, g_gamma, &dp, &variant, &smem, &tab);
    const bool gen3 = variant >= kNumVariants2;
    const Variant3 v3 = gen3 ? kVariants3[variant - kNumVariants2] : Variant3{0, 0, 0, 0, 0, 0, 0, 0};
    const int64_t vals[17] = {variant, gen3 ? v3.DEG : 0, gen3 ? v3.NWE : 0, gen3 ? v3.NG : 0, gen3 ? v3.NJA : 0,
                              gen3 ? v3.NJB : 0, dp.HS, dp.WZ, dp.Sy, dp.Sz, dp.Hy, dp.Hz, dp.chunk, (int64_t)smem,
                              dp.t_max >= 0.f, dp.nr_min, dp.nr_max};
    for (int i = 0; i < 17; ++i) out[i] = vals[i];
    if (task_table_host)
        for (int64_t i = 0; i < std::min<int64_t>(table_cap, (int64_t)tab.size()); ++i) task_table_host[i] = tab[(size_t)i];
    return (int64_t)tab.size();
}

int jpet_abi_version(void) { return JPET_ABI_VERSION; }

}  // extern "C"
