// rows_launch.h - host-side interface between the API (jpet_api.cu) and the instantiations of the tiled event kernel
// (rows_inst.cu, compiled once per group of shapes so that build.py can run the groups in parallel).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <string>

#include "common.cuh"

namespace jpet_host {

// Shapes of the tiled event kernel (mlem_rows.cuh): NWE warps per event, NG event groups per CTA, NJA / NJB pixel capacity
// of the two pieces a lane walks (NJB = 0: one piece), region row stride HS, MINB resident CTAs per SM asked of the
// compiler, DEG: 0 = closed form (rsqrt + ex2 per pixel), 4 / 5 = exponent as a polynomial in u (one ex2 per pixel;
// make_plan bounds the truncation error and picks the degree), BW: pixels per block of the walks.  Ordered by size
// within each degree: make_plan takes the first one of the wanted degree that holds the workload's ellipses.  The
// last column is the compilation group.  Block widths are the measured optima of round 1.
// CLS = 1: the instance can walk one degree class of a two-class sort (mlem_rows.cuh); 0 keeps the one-class item loop
// (the 44- and 52-pixel shapes sit at their register limit: the extra bookkeeping costs them 1.4 %).
//        name          NWE NG NJA NJB  HS MINB DEG BW CLS group
#define JPET_SHAPES(X)                                                                                              \
    X(small_closed,      1, 4, 12,  0,  64, 4,  0, 16, 0, 0) /* <= 32 rows, chords <= 12 px           (fig4)        */ \
    X(mid_closed,        1, 4, 20,  8,  64, 4,  0,  8, 0, 0) /* <= 64 rows, chords <= 20 px                         */ \
    X(large_closed,      4, 4, 36,  0, 128, 1,  0,  8, 0, 0) /* <= 128 rows, chords <= 36 px, four warps per event  */ \
    X(xl_closed,         4, 4, 44,  0, 128, 1,  0,  8, 0, 0) /* <= 128 rows, chords <= 44 px                        */ \
    X(xxl_closed,        4, 3, 52,  0, 128, 1,  0,  8, 0, 0) /* <= 128 rows, chords <= 52 px, three groups (168 registers) */ \
    X(small_deg3,        1, 4, 12,  0,  64, 4,  3,  8, 1, 0) /* degree 3: where the plan's bound allows it (config 3), and for   */ \
    X(mid18_deg3,        1, 4, 18,  8,  64, 4,  3, 32, 1, 2) /* the events of degree class 1 of a degree-4 / 5 plan (make_plan) */ \
    X(mid_deg3,          1, 4, 20,  8,  64, 4,  3, 32, 1, 0)                                                          \
    X(large_deg3,        4, 4, 36,  0, 128, 1,  3, 16, 1, 2)                                                          \
    X(small_deg4,        1, 4, 12,  0,  64, 4,  4,  8, 1, 1) /*                                       (config 1)    */ \
    X(mid18_deg4,        1, 4, 18,  8,  64, 4,  4, 32, 1, 3) /* one block per piece, chords <= 18 px   (config 2)    */ \
    X(mid_deg4,          1, 4, 20,  8,  64, 4,  4, 32, 1, 1) /* one block per piece                                  */ \
    X(large_deg4,        4, 4, 36,  0, 128, 1,  4, 16, 1, 1) /*                                       (config 4)    */ \
    X(xl_deg4,           4, 4, 44,  0, 128, 1,  4, 16, 0, 1) /*                                       (config 5)    */ \
    X(xxl_deg4,          4, 3, 52,  0, 128, 1,  4, 16, 0, 1) /* (config 5 with a position-dependent sigma_z)        */ \
    X(small_deg5,        1, 4, 12,  0,  64, 4,  5,  8, 1, 2)                                                          \
    X(mid_deg5,          1, 4, 20,  8,  64, 4,  5,  8, 1, 2)                                                          \
    X(large_deg5,        4, 4, 36,  0, 128, 1,  5, 16, 1, 2)                                                          \
    X(xl_deg5,           4, 4, 44,  0, 128, 1,  5,  8, 0, 3)                                                          \
    X(xxl_deg5,          4, 3, 52,  0, 128, 1,  5, 16, 0, 3)

struct Shape { const char* name; int NWE, NG, NJA, NJB, HS, MINB, DEG, BW, CLS; };

enum ShapeId {
#define JPET_X(name, NWE, NG, NJA, NJB, HS, MINB, DEG, BW, CLS, GRP) k_##name,
    JPET_SHAPES(JPET_X)
#undef JPET_X
    kNumShapes
};

constexpr Shape kShapes[] = {
#define JPET_X(name, NWE, NG, NJA, NJB, HS, MINB, DEG, BW, CLS, GRP) {#name, NWE, NG, NJA, NJB, HS, MINB, DEG, BW, CLS},
    JPET_SHAPES(JPET_X)
#undef JPET_X
};
constexpr int kNumGroups = 4;

// One batch of events sorted by sub-tile, with its work-item list (device memory).
struct BinSet {
    float* sorted = nullptr;            // EventRec [n] (16 floats each), regular bins first, the direct bin last
    jpet::WorkItem* items = nullptr;
    int* meta = nullptr;                // jpet::MetaWord (common.cuh)
    int64_t n = 0;
    size_t cap_events = 0, cap_items = 0;
    bool owns_sorted = true;
};

struct RowsPlan {
    jpet::DevParams dp{};
    int shape = 0;
    int shape_lo = -1;                  // >= 0: the degree-3 instance of `shape` for the events of degree class 1 (dp.n_cls == 2)
    size_t smem = 0;
    bool vs = false;                    // sigma_z depends on the hit positions (kernel template flag VS)
};

struct RowsLaunch {
    const BinSet* bs;
    const RowsPlan* plan;
    const float* wT;
    float* accT;
    const uint32_t* tab;
    unsigned long long* counters;
    int sm_count, device, ctas_per_sm;
    int shape, cls;                     // which shape to launch over which degree class
    int64_t max_items;
    cudaStream_t stream;
    bool pdl;
};

// Launches the tiled event kernel of plan->shape (JPET_OK or an error code with the text set).
int launch_rows_shape(const RowsLaunch& rl);
// One per compilation group: returns -100 when the shape is not in the group.
int launch_rows_group0(const RowsLaunch& rl);
int launch_rows_group1(const RowsLaunch& rl);
int launch_rows_group2(const RowsLaunch& rl);
int launch_rows_group3(const RowsLaunch& rl);

extern std::atomic<uint64_t> g_launches;
extern thread_local std::string g_err;
int fail(int code, const char* fmt, ...);

}  // namespace jpet_host
