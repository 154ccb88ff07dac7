// rows_inst.cu - instantiations of the tiled event kernel for one group of shapes (-DJPET_GROUP=g; build.py compiles
// the groups in parallel) and their launch code.
#include "../../include/jpet.h"
#include "mlem_rows.cuh"
#include "rows_launch.h"

#ifndef JPET_GROUP
#error "compile with -DJPET_GROUP=<0..3>"
#endif

namespace jpet_host {
namespace {

#define CUDA_TRY(expr)                                                                              \
    do {                                                                                            \
        cudaError_t _e = (expr);                                                                    \
        if (_e != cudaSuccess) {                                                                    \
            (void)cudaGetLastError(); /* reported here: do not leave it for an unrelated later call */ \
            return fail(JPET_E_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(_e), __FILE__, __LINE__); \
        }                                                                                           \
    } while (0)

// Persistent grid: resident CTAs per SM x SMs (capped by the number of work items); launched with programmatic stream
// serialisation (the kernel starts with pdl_wait()).
template <int NWE, int NG, int NJA, int NJB, int HS, int MINB, int DEG, int BW, bool VS, bool CLS>
int launch_rows(const RowsLaunch& rl) {
    constexpr int NT = NWE * NG * 32;
    auto kern = jpet::mlem_rows_kernel<NWE, NG, NJA, NJB, HS, MINB, DEG, BW, VS, CLS>;
    if (!CLS && (rl.cls != 0 || rl.plan->dp.n_cls != 1)) return fail(JPET_E_INVAL, "internal: shape without degree classes launched on a two-class sort");
    const jpet::DevParams& dp = rl.plan->dp;
    const size_t smem = rl.plan->smem;
    if (dp.HS != HS) return fail(JPET_E_INVAL, "internal: region stride %d does not match the kernel's %d", dp.HS, HS);
    static size_t attr_set[64] = {};                       // per device: the attribute belongs to the device's copy of the function
    if (rl.device < 0 || rl.device >= 64) return fail(JPET_E_INVAL, "device ordinal out of range");
    if (smem > 40 * 1024 && smem > attr_set[rl.device]) {
        CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set[rl.device] = smem;
    }
    int per_sm = 0;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem));
    if (per_sm < 1) return fail(JPET_E_CUDA, "event kernel does not fit on an SM (%zu B of shared memory)", smem);
    if (rl.ctas_per_sm > 0) per_sm = std::min(per_sm, rl.ctas_per_sm);
    const int grid = (int)std::min<int64_t>((int64_t)rl.sm_count * per_sm, std::max<int64_t>(rl.max_items, 1));
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(NT);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = rl.stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = rl.pdl ? 1 : 0;
    CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, reinterpret_cast<const jpet::EventRec*>(rl.bs->sorted), (const jpet::WorkItem*)rl.bs->items,
                                rl.bs->meta, dp, rl.wT, rl.accT, rl.tab, rl.counters, rl.cls));
    g_launches++;
    CUDA_TRY(cudaGetLastError());
    return JPET_OK;
}

}  // namespace

#define JPET_CAT2(a, b) a##b
#define JPET_CAT(a, b) JPET_CAT2(a, b)

int JPET_CAT(launch_rows_group, JPET_GROUP)(const RowsLaunch& rl) {
    switch (rl.shape) {
#define JPET_X(name, NWE, NG, NJA, NJB, HS, MINB, DEG, BW, CLS, GRP)                                         \
    case k_##name:                                                                                           \
        if constexpr (GRP == JPET_GROUP)                                                                     \
            return rl.plan->vs ? launch_rows<NWE, NG, NJA, NJB, HS, MINB, DEG, BW, true, CLS != 0>(rl)       \
                               : launch_rows<NWE, NG, NJA, NJB, HS, MINB, DEG, BW, false, CLS != 0>(rl);     \
        else return -100;
        JPET_SHAPES(JPET_X)
#undef JPET_X
        default: return -100;
    }
}

}  // namespace jpet_host
