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
//        name          NWE NG NJA NJB  HS MINB DEG BW  group
#define JPET_SHAPES(X)                                                                                              \
    X(small_closed,      1, 4, 12,  0,  64, 4,  0, 16,  0) /* <= 32 rows, chords <= 12 px           (fig4)        */ \
    X(mid_closed,        1, 4, 20,  8,  64, 4,  0,  8,  0) /* <= 64 rows, chords <= 20 px                         */ \
    X(large_closed,      4, 4, 36,  0, 128, 1,  0,  8,  0) /* <= 128 rows, chords <= 36 px, four warps per event  */ \
    X(xl_closed,         4, 4, 44,  0, 128, 1,  0,  8,  0) /* <= 128 rows, chords <= 44 px                        */ \
    X(xxl_closed,        4, 3, 52,  0, 128, 1,  0,  8,  0) /* <= 128 rows, chords <= 52 px, three groups (168 registers) */ \
    X(small_deg4,        1, 4, 12,  0,  64, 4,  4,  8,  1) /*                                       (config 1)    */ \
    X(mid18_deg4,        1, 4, 18,  8,  64, 4,  4, 32,  3) /* one block per piece, chords <= 18 px   (configs 2, 3) */ \
    X(mid_deg4,          1, 4, 20,  8,  64, 4,  4, 32,  1) /* one block per piece                                  */ \
    X(large_deg4,        4, 4, 36,  0, 128, 1,  4, 16,  1) /*                                       (config 4)    */ \
    X(xl_deg4,           4, 4, 44,  0, 128, 1,  4, 16,  1) /*                                       (config 5)    */ \
    X(xxl_deg4,          4, 3, 52,  0, 128, 1,  4, 16,  1) /* (config 5 with a position-dependent sigma_z)        */ \
    X(small_deg5,        1, 4, 12,  0,  64, 4,  5,  8,  2)                                                          \
    X(mid_deg5,          1, 4, 20,  8,  64, 4,  5,  8,  2)                                                          \
    X(large_deg5,        4, 4, 36,  0, 128, 1,  5, 16,  2)                                                          \
    X(xl_deg5,           4, 4, 44,  0, 128, 1,  5,  8,  3)                                                          \
    X(xxl_deg5,          4, 3, 52,  0, 128, 1,  5, 16,  3)

struct Shape { const char* name; int NWE, NG, NJA, NJB, HS, MINB, DEG, BW; };

enum ShapeId {
#define JPET_X(name, NWE, NG, NJA, NJB, HS, MINB, DEG, BW, GRP) k_##name,
    JPET_SHAPES(JPET_X)
#undef JPET_X
    kNumShapes
};

constexpr Shape kShapes[] = {
#define JPET_X(name, NWE, NG, NJA, NJB, HS, MINB, DEG, BW, GRP) {#name, NWE, NG, NJA, NJB, HS, MINB, DEG, BW},
    JPET_SHAPES(JPET_X)
#undef JPET_X
};
constexpr int kNumGroups = 4;

// One batch of events sorted by sub-tile, with its work-item list (device memory).
struct BinSet {
    float* sorted = nullptr;            // EventRec [n] (16 floats each), regular bins first, the direct bin last
    jpet::WorkItem* items = nullptr;
    int* meta = nullptr;                // 0: #items, 1: direct start, 2: direct count, 3: work counter
    int64_t n = 0;
    size_t cap_events = 0, cap_items = 0;
    bool owns_sorted = true;
};

struct RowsPlan {
    jpet::DevParams dp{};
    int shape = 0;
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
