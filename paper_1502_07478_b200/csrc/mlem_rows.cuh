// mlem_rows.cuh - the tiled event kernel of the list-mode MLEM hot path (sm_100a): steps 1-3 of an iteration for the
// events of the regular bins - ellipse rows and spans (App. B :251-267), the kernel of Eq. 7-12
// with the denominator of Eq. 3, and the back-projection (Listing 1 line 10).
//
// Design (B200, not the paper's warp-per-event / texture scheme):
//   * events are pre-sorted by image sub-tile (sort_kernels.cuh) and carry a 64-byte record of per-event constants; a
//     CTA takes a work item (sub-tile, chunk of events), stages the w = s*rho region (sub-tile + halo) in shared
//     memory, accumulates P / denominator into PRIVATE shared-memory regions with plain (non-atomic) read-modify-
//     writes, and flushes them once with red.global.add.f32 (measured: global red.add tops out at ~2.8e10 warp
//     requests/s, a factor 5-10 below what the SFU/FP32 pipes produce, so the scatter has to stay on chip);
//   * regions are stored transposed (y fastest, row stride HS a multiple of 32): lanes are consecutive image rows, so
//     whole-row pieces of a warp never share a bank whatever the ellipse tilt (split cap rows do: see piece B);
//   * an event is handled by a GROUP of NWE warps (1 for ellipses of up to 64 rows), several groups per CTA share one
//     staged w region and own one accumulator region each; with NWE = 1 the event loop has no barrier at all (the
//     denominator is a warp shuffle reduction);
//   * every lane owns up to two PIECES of ellipse rows per event: piece A, a whole row of the central block
//     (capacity NJA pixels), and piece B, a row or a half / quarter of a row of the caps (capacity NJB).  Which
//     (row, part) a lane takes is read from a table indexed by the number of rows of the ellipse, built on
//     the host from the ellipse geometry (task_table.h) and kept in shared memory - no index arithmetic;
//   * the row constants of the two pieces are evaluated together in packed fp32x2 arithmetic; the kernel values of a
//     piece stay in registers between the denominator pass and the back-projection pass;
//   * pixel walks are cut into blocks of BW pixels entered through one warp-uniform switch, pairs of pixels per fp32x2
//     operation; the ragged ends of the rows are masked per pixel;
//   * DEG > 0: the exponent of Eq. 7 as a degree-DEG polynomial in u along a piece (poly_coeffs2): one ex2 per kernel
//     value instead of rsqrt + ex2, the Horner steps of all pairs of a block in lockstep;
//   * the back-projection pass issues its shared-memory read-modify-writes eight at a time; when every lane of a
//     one-warp group owns at least 8 pixels of its central row, the first 8 run without masks and predicates;
//   * VS: sigma_z depends on the hit positions (common.cuh): the Gaussian coefficient GS and the chord H0p / GS are
//     per event;
//   * every kernel of an iteration starts with pdl_wait() and is launched with programmatic stream serialisation.
//
// Citations are /root/reference/PAPER.md lines.  Nothing here is shared with oracle/.
#pragma once
#include "common.cuh"

namespace jpet {

// Table: one 32-bit word per (row count of the ellipse, lane of the group): piece A in bits 0-15, piece B in bits
// 16-31.  A 16-bit entry: bits 0-7 row (relative to the first row of the unclipped ellipse), 8-9 part,
// 10-11 log2(parts), bit 15 valid.  Slot A only ever holds whole rows.
constexpr uint32_t kTaskValid = 1u << 15;

__device__ __forceinline__ f32x2 bc2(float x) { return pack2(x, x); }

struct Piece {
    RowWalk rc;          // rc.lo / rc.len: first column and pixel count of the piece
    uint32_t off;        // byte offset of its first pixel inside a region
    float c[6];          // DEG > 0: log2 P = c[0] + c[1] v + ... + c[DEG] v^DEG along the piece (see poly_coeffs2)
    float ngs;           // DEG = 0: -GS, the coefficient of the Gaussian term (-1 for a constant sigma_z)
};

__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2_approx(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// One MUFU per kernel value instead of two.  Along a row (v = scaled u, common.cuh) Eq. 7 reads
//     log2 P = c2s - v^2 + ba(v)^2 / D(v) - 1/2 log2 D(v),     ba = alphas v + betas,   D = delta + eps v,
// and x = eps v / delta is small inside the 3-sigma ellipse: |x| <= 2 |t| |y| |u| / (sec^2 (R^2 + y^2)), a few
// per cent at most (the host plan bounds it and picks DEG, or falls back to DEG = 0, the closed form).  With
// kappa = eps / delta, 1 / D = (1 - x + x^2 - ...) / delta and ln D = ln delta + x - x^2/2 + x^3/3 - ..., so
//     ba^2 / D = sum_n e_n v^n,   e_0 = beta^2 / delta,  e_1 = 2 alpha beta / delta - kappa e_0,
//                                 e_2 = alpha^2 / delta - kappa e_1,  e_n = -kappa e_(n-1)  (n >= 3),
//     -1/2 log2 D = -1/2 log2 delta - LH (kappa v - kappa^2 v^2 / 2 + kappa^3 v^3 / 3 - ...),   LH = log2(e) / 2.
// The series is cut after v^DEG; the neglected terms are bounded by (ba^2/D) |x|^(DEG-1) + |x|^(DEG+1).
// Two pieces (A in the low half, B in the high half) at a time.
// NGS = -GS: coefficient of the Gaussian term (-1 for a constant sigma_z).
template <int DEG>
__device__ __forceinline__ void poly_coeffs2(f32x2 C2S, f32x2 BET, f32x2 ALP, f32x2 EPS, f32x2 DEL, float NGS, f32x2 (&C)[6]) {
    float d0, d1;
    unpack2(DEL, d0, d1);
    const f32x2 G = pack2(rcp_approx(d0), rcp_approx(d1));
    const f32x2 L2 = pack2(lg2_approx(d0), lg2_approx(d1));
    const f32x2 NK = mul2(mul2(EPS, G), bc2(-1.f));                   // -kappa
    const f32x2 GB = mul2(G, BET), GA = mul2(G, ALP);
    f32x2 E[6], K[6];
    E[0] = mul2(GB, BET);
    E[1] = fma2(NK, E[0], mul2(add2(GB, GB), ALP));
    E[2] = fma2(NK, E[1], mul2(GA, ALP));
    K[1] = NK;                                                          // K[n] = (-kappa)^n
#pragma unroll
    for (int n = 2; n <= DEG; ++n) K[n] = mul2(K[n - 1], NK);
#pragma unroll
    for (int n = 3; n <= DEG; ++n) E[n] = mul2(NK, E[n - 1]);
    C[0] = fma2(L2, bc2(-0.5f), add2(C2S, E[0]));
    C[1] = fma2(K[1], bc2(kLH), E[1]);                                  // -LH kappa
    C[2] = fma2(K[2], bc2(0.5f * kLH), add2(E[2], bc2(NGS)));           // +LH kappa^2 / 2, and the Gaussian -GS v^2
#pragma unroll
    for (int n = 3; n <= DEG; ++n) C[n] = fma2(K[n], bc2(kLH / (float)n), E[n]);      // (-1)^n LH kappa^n / n
}

// Span of one piece: row iy (valid or not), half chord^2 hw2 [px^2], chord centre zcp [px]; part `part` of 2^sh.
template <int CAP, int HS, bool SPLIT>
__device__ __forceinline__ void piece_span(uint32_t te, int iy, float hw2, float zcp, float pxs, const DevParams& p, int ry0,
                                           int rz0, int col_lo, int col_hi, Piece& pc, int& overflow) {
    const bool valid = (te & kTaskValid) && (unsigned)iy < (unsigned)p.n_y && hw2 >= 0.f;
    const float hw = sqrt_approx(fmaxf(hw2, 0.f));
    int lo = max(col_lo, __float2int_ru(zcp - hw));
    const int hi = min(col_hi, __float2int_rd(zcp + hw));
    int len = valid ? max(0, hi - lo + 1) : 0;
    if constexpr (SPLIT) {
        const int part = (te >> 8) & 3, sh = (te >> 10) & 3;
        const int plen = (len + (1 << sh) - 1) >> sh;
        const int first = min(len, part * plen);
        len = min(len - first, plen);
        lo += first;
    }
    overflow |= len > CAP;
    len = min(len, CAP);                       // never taken: the table guarantees the capacity (task_table.h)
    if (len == 0) { lo = rz0; iy = ry0; pc.rc.delta = 1.f; pc.rc.eps = 0.f; }     // idle lanes stay inside the region
    pc.rc.u0s = ((float)lo - zcp) * pxs;
    pc.rc.lo = lo;
    pc.rc.len = len;
    pc.off = 4u * (uint32_t)((lo - rz0) * HS + (iy - ry0));
}

// Row constants of pieces A and B (polynomials in dy, see EventRec in common.cuh) in packed arithmetic, then their spans.
template <int NJA, int NJB, int HS, int DEG, bool VS>
__device__ __forceinline__ void pieces_setup(uint32_t te, const float4 r0, const float4 r1, const float4 r2,
                                             const float4 r3, const DevParams& p, int ry0, int rz0, int col_lo, int col_hi,
                                             Piece& A, Piece& B, int& overflow) {
    const int iy0 = rows_first(__float_as_int(r3.w));
    const float ngs = VS ? -r3.z : -1.f;                               // -GS
    const float H0e = VS ? p.H0p * rcp_approx(r3.z) : p.H0p;            // half chord^2 at the centre row [px^2]
    const uint32_t teA = te, teB = te >> 16;
    const int iyA = iy0 + (int)(teA & 0xffu), iyB = iy0 + (int)(teB & 0xffu);
    if constexpr (NJB > 0) {
        const f32x2 DY = fma2(pack2((float)iyA, (float)iyB), bc2(p.px), bc2(r0.x));
        const f32x2 DY2 = mul2(DY, DY);
        const f32x2 C2S = mul2(bc2(r0.y), DY2);
        const f32x2 BET = mul2(DY, fma2(bc2(r0.w), DY, bc2(r0.z)));
        const f32x2 ALP = fma2(bc2(r1.y), DY, bc2(r1.x));
        const f32x2 EPS = fma2(bc2(r1.w), DY, bc2(r1.z));
        const f32x2 DEL = fma2(DY, fma2(bc2(r2.z), DY, bc2(r2.y)), bc2(r2.x));
        const f32x2 HW2 = fma2(bc2(r2.w), DY2, bc2(H0e));
        const f32x2 ZCP = fma2(bc2(r3.y), DY, bc2(r3.x));
        float hwA, hwB, zcA, zcB;
        unpack2(C2S, A.rc.c2s, B.rc.c2s);
        unpack2(BET, A.rc.betas, B.rc.betas);
        unpack2(ALP, A.rc.alphas, B.rc.alphas);
        unpack2(EPS, A.rc.eps, B.rc.eps);
        unpack2(DEL, A.rc.delta, B.rc.delta);
        unpack2(HW2, hwA, hwB);
        unpack2(ZCP, zcA, zcB);
        A.ngs = B.ngs = ngs;
        if constexpr (DEG > 0) {
            f32x2 C[6];
            poly_coeffs2<DEG>(C2S, BET, ALP, EPS, DEL, ngs, C);
#pragma unroll
            for (int n = 0; n <= DEG; ++n) unpack2(C[n], A.c[n], B.c[n]);
        }
        piece_span<NJA, HS, false>(teA, iyA, hwA, zcA, p.pxs, p, ry0, rz0, col_lo, col_hi, A, overflow);
        piece_span<NJB, HS, true>(teB, iyB, hwB, zcB, p.pxs, p, ry0, rz0, col_lo, col_hi, B, overflow);
    } else {
        const float dy = fmaf((float)iyA, p.px, r0.x);
        const float dy2 = dy * dy;
        A.rc.c2s = r0.y * dy2;
        A.rc.betas = dy * fmaf(r0.w, dy, r0.z);
        A.rc.alphas = fmaf(r1.y, dy, r1.x);
        A.rc.eps = fmaf(r1.w, dy, r1.z);
        A.rc.delta = fmaf(dy, fmaf(r2.z, dy, r2.y), r2.x);
        A.ngs = ngs;
        if constexpr (DEG > 0) {
            f32x2 C[6];
            poly_coeffs2<DEG>(bc2(A.rc.c2s), bc2(A.rc.betas), bc2(A.rc.alphas), bc2(A.rc.eps), bc2(A.rc.delta), ngs, C);
            float dummy;
#pragma unroll
            for (int n = 0; n <= DEG; ++n) unpack2(C[n], A.c[n], dummy);
        }
        piece_span<NJA, HS, false>(teA, iyA, fmaf(r2.w, dy2, H0e), fmaf(r3.y, dy, r3.x), p.pxs, p, ry0, rz0, col_lo, col_hi, A, overflow);
    }
}

// State of one pixel walk (pass 1): packed row constants, running u' pair and denominator pair.
struct Walk {
    f32x2 EPS2, DEL2, ALP2, BET2, C2S2, NGS2, STEP2, V2, DEN2;
    f32x2 C[6];          // DEG > 0: broadcast polynomial coefficients (EPS2 ... C2S2 unused)
    uint32_t wa;
    int len;
};

// Two adjacent pixels j, j+1 of the piece: Eq. 7 (up to the constant K) and the denominator term.
template <int J, int HS, bool MASK, int DEG, bool VS>
__device__ __forceinline__ void walk_pair(Walk& s, float& p0, float& p1) {
    if constexpr (DEG > 0) {
        f32x2 E2 = fma2(s.C[DEG], s.V2, s.C[DEG - 1]);
#pragma unroll
        for (int n = DEG - 2; n >= 0; --n) E2 = fma2(E2, s.V2, s.C[n]);
        float e0, e1;
        unpack2(E2, e0, e1);
        float x0 = ex2_approx(e0), x1 = ex2_approx(e1);
        if (MASK) {
            x0 = J < s.len ? x0 : 0.f;
            x1 = J + 1 < s.len ? x1 : 0.f;
        }
        s.DEN2 = fma2(pack2(x0, x1), pack2(lds_imm<4 * J * HS>(s.wa), lds_imm<4 * (J + 1) * HS>(s.wa)), s.DEN2);
        p0 = x0;
        p1 = x1;
        s.V2 = add2(s.V2, s.STEP2);
        return;
    }
    const f32x2 D2 = fma2(s.EPS2, s.V2, s.DEL2), BA2 = fma2(s.ALP2, s.V2, s.BET2);
    float d0, d1;
    unpack2(D2, d0, d1);
    const f32x2 RS2 = pack2(rsqrt_approx(d0), rsqrt_approx(d1));
    const f32x2 BAR2 = mul2(BA2, RS2);
    f32x2 E2;
    if constexpr (VS) E2 = fma2(mul2(s.NGS2, s.V2), s.V2, fma2(BAR2, BAR2, s.C2S2));     // c2s - GS v^2 + bar^2
    else E2 = fma2(add2(BAR2, s.V2), sub2(BAR2, s.V2), s.C2S2);                           // c2s - v^2 + bar^2
    float e0, e1;
    unpack2(E2, e0, e1);
    float x0 = ex2_approx(e0), x1 = ex2_approx(e1);
    if (MASK) {
        x0 = J < s.len ? x0 : 0.f;
        x1 = J + 1 < s.len ? x1 : 0.f;
    }
    const f32x2 P2 = mul2(RS2, pack2(x0, x1));
    s.DEN2 = fma2(P2, pack2(lds_imm<4 * J * HS>(s.wa), lds_imm<4 * (J + 1) * HS>(s.wa)), s.DEN2);
    unpack2(P2, p0, p1);
    s.V2 = add2(s.V2, s.STEP2);
}

// Pixel walks are cut into blocks of BW pixels entered through ONE switch on the number of blocks the warp needs
// (highest block first, falling through to block 0): no compare-and-branch between blocks - ncu showed each such
// pair to cost the 4-warp schedulers about as much as the block's own arithmetic - and every block is one basic
// block of BW / 2 independent pixel pairs for the scheduler to interleave.  All pairs are masked by the lane's own
// pixel count.
// BW (template parameter): pixels per block - 8, 16 or 32 in the shipped shapes (rows_launch.h).

// DEG > 0: the pairs of a block in LOCKSTEP - all u' pairs, then one Horner step for every pair, ..., then the ex2, the
// masks and the denominator terms (two accumulators).  ptxas keeps source order: written pair after pair it issued the
// four dependent FFMA2 of a Horner chain back to back (4-cycle waits, the largest stall of the kernel in ncu).
// NFULL: the first NFULL pixels of the block belong to the chord in EVERY lane of the warp (no masks for them).
template <int JB, int NJ, int HS, int DEG, int BW, int NFULL = 0>
__device__ __forceinline__ void walk_block_lockstep(Walk& s, float u0s, float pxs, float (&preg)[NJ]) {
    constexpr int NPAIR = (NJ - JB < BW ? NJ - JB : BW) / 2;
    const float vb = fmaf((float)JB, pxs, u0s);
    f32x2 V[NPAIR], E[NPAIR];
    float x[2 * NPAIR];
    V[0] = pack2(vb, vb + pxs);
#pragma unroll
    for (int k = 1; k < NPAIR; ++k) V[k] = add2(V[k - 1], s.STEP2);
#pragma unroll
    for (int k = 0; k < NPAIR; ++k) E[k] = fma2(s.C[DEG], V[k], s.C[DEG - 1]);
#pragma unroll
    for (int n = DEG - 2; n >= 0; --n) {
#pragma unroll
        for (int k = 0; k < NPAIR; ++k) E[k] = fma2(E[k], V[k], s.C[n]);
    }
#pragma unroll
    for (int k = 0; k < NPAIR; ++k) {
        float e0, e1;
        unpack2(E[k], e0, e1);
        x[2 * k] = ex2_approx(e0);
        x[2 * k + 1] = ex2_approx(e1);
    }
    f32x2 DENB = pack2(0.f, 0.f);
    static_for<0, NPAIR>([&](auto kc) {
        constexpr int K = decltype(kc)::value, J = JB + 2 * K;
        float x0 = x[2 * K], x1 = x[2 * K + 1];
        if constexpr (J - JB >= NFULL) x0 = J < s.len ? x0 : 0.f;
        if constexpr (J + 1 - JB >= NFULL) x1 = J + 1 < s.len ? x1 : 0.f;
        const f32x2 W2 = pack2(lds_imm<4 * J * HS>(s.wa), lds_imm<4 * (J + 1) * HS>(s.wa));
        if constexpr (K & 1) DENB = fma2(pack2(x0, x1), W2, DENB);
        else s.DEN2 = fma2(pack2(x0, x1), W2, s.DEN2);
        preg[J] = x0;
        preg[J + 1] = x1;
    });
    if constexpr (NPAIR > 1) s.DEN2 = add2(s.DEN2, DENB);
}

template <int JB, int NJ, int HS, int DEG, int BW, bool VS, int NFULL = 0>
__device__ __forceinline__ void walk_block(Walk& s, float u0s, float pxs, float (&preg)[NJ]) {
    if constexpr (DEG > 0) {
        if constexpr (JB < NJ) walk_block_lockstep<JB, NJ, HS, DEG, BW, NFULL>(s, u0s, pxs, preg);
    } else {
        const float vb = fmaf((float)JB, pxs, u0s);
        s.V2 = pack2(vb, vb + pxs);
        static_for<0, BW / 2>([&](auto kc) {
            constexpr int J = JB + 2 * decltype(kc)::value;
            if constexpr (J < NJ) walk_pair<J, HS, true, DEG, VS>(s, preg[J], preg[J + 1]);
        });
    }
}

#define JPET_BLOCK_CASES(CALL)                                                 \
    switch (nblk) {                                                            \
        default:                                                               \
        case 12: if constexpr (NB > 11) { CALL(11); } [[fallthrough]];         \
        case 11: if constexpr (NB > 10) { CALL(10); } [[fallthrough]];         \
        case 10: if constexpr (NB > 9) { CALL(9); } [[fallthrough]];           \
        case 9: if constexpr (NB > 8) { CALL(8); } [[fallthrough]];            \
        case 8: if constexpr (NB > 7) { CALL(7); } [[fallthrough]];            \
        case 7: if constexpr (NB > 6) { CALL(6); } [[fallthrough]];            \
        case 6: if constexpr (NB > 5) { CALL(5); } [[fallthrough]];            \
        case 5: if constexpr (NB > 4) { CALL(4); } [[fallthrough]];            \
        case 4: if constexpr (NB > 3) { CALL(3); } [[fallthrough]];            \
        case 3: if constexpr (NB > 2) { CALL(2); } [[fallthrough]];            \
        case 2: if constexpr (NB > 1) { CALL(1); } [[fallthrough]];            \
        case 1: { CALL(0); } [[fallthrough]];                                  \
        case 0: break;                                                         \
    }

// full8 (warp-uniform): every lane of the warp has at least 8 pixels, so block 0 runs its first 8 pixels without masks.
template <int NJ, int HS, int DEG, int BW, bool VS>
__device__ __forceinline__ float piece_pass1(const Piece& pc, uint32_t w_addr, float pxs, int nblk, float (&preg)[NJ],
                                             bool full8 = false) {
    static_assert(NJ % 2 == 0 && NJ <= 12 * BW && (BW == 4 || BW == 8 || BW == 16 || BW == 32), "pixel capacity must be even and at most 12 blocks");
    constexpr int NB = (NJ + BW - 1) / BW;
    Walk s;
    if constexpr (DEG > 0) {
#pragma unroll
        for (int n = 0; n <= DEG; ++n) s.C[n] = bc2(pc.c[n]);
    } else {
        s.EPS2 = bc2(pc.rc.eps); s.DEL2 = bc2(pc.rc.delta); s.ALP2 = bc2(pc.rc.alphas); s.BET2 = bc2(pc.rc.betas);
        s.C2S2 = bc2(pc.rc.c2s);
        s.NGS2 = bc2(pc.ngs);
    }
    s.STEP2 = bc2(2.f * pxs);
    s.DEN2 = pack2(0.f, 0.f);
    s.wa = w_addr + pc.off;
    s.len = pc.rc.len;
    const float u0s = pc.rc.u0s;
#define JPET_WALK(B)                                                                          \
    do {                                                                                      \
        if ((B) == 0 && DEG > 0 && BW >= 8 && NJ >= 8 && full8) walk_block<0, NJ, HS, DEG, BW, VS, 8>(s, u0s, pxs, preg); \
        else walk_block<(B) * BW, NJ, HS, DEG, BW, VS>(s, u0s, pxs, preg);                    \
    } while (0)
    JPET_BLOCK_CASES(JPET_WALK)
#undef JPET_WALK
    float q0, q1;
    unpack2(s.DEN2, q0, q1);
    return q0 + q1;
}

// acc[addr + IMM + k STRIDE] += P_k * inv for k = 0..3, lanes with len > J + k: four loads in flight, then the four
// multiply-adds, then the stores (one asm block so that the loads are not serialised behind the previous store).
template <int IMM, int STRIDE, int J>
__device__ __forceinline__ void smem_fma_if4(uint32_t addr, float P0, float P1, float P2, float P3, float inv, int len) {
    asm volatile(
        "{\n\t.reg .pred p0, p1, p2, p3;\n\t.reg .f32 t0, t1, t2, t3;\n\t"
        "setp.gt.s32 p0, %6, %7;\n\t"
        "setp.gt.s32 p1, %6, %8;\n\t"
        "setp.gt.s32 p2, %6, %9;\n\t"
        "setp.gt.s32 p3, %6, %10;\n\t"
        "@p0 ld.shared.f32 t0, [%0 + %11];\n\t"
        "@p1 ld.shared.f32 t1, [%0 + %12];\n\t"
        "@p2 ld.shared.f32 t2, [%0 + %13];\n\t"
        "@p3 ld.shared.f32 t3, [%0 + %14];\n\t"
        "@p0 fma.rn.f32 t0, %1, %5, t0;\n\t"
        "@p1 fma.rn.f32 t1, %2, %5, t1;\n\t"
        "@p2 fma.rn.f32 t2, %3, %5, t2;\n\t"
        "@p3 fma.rn.f32 t3, %4, %5, t3;\n\t"
        "@p0 st.shared.f32 [%0 + %11], t0;\n\t"
        "@p1 st.shared.f32 [%0 + %12], t1;\n\t"
        "@p2 st.shared.f32 [%0 + %13], t2;\n\t"
        "@p3 st.shared.f32 [%0 + %14], t3;\n\t}"
        ::"r"(addr), "f"(P0), "f"(P1), "f"(P2), "f"(P3), "f"(inv), "r"(len), "n"(J), "n"(J + 1), "n"(J + 2), "n"(J + 3),
          "n"(IMM), "n"(IMM + STRIDE), "n"(IMM + 2 * STRIDE), "n"(IMM + 3 * STRIDE)
        : "memory");
}

// Eight at a time (blocks of 8 or 16 pixels): eight loads in flight before the first multiply-add.
template <int IMM, int STRIDE, int J>
__device__ __forceinline__ void smem_fma_if8(uint32_t addr, const float* P, float inv, int len) {
    asm volatile(
        "{\n\t.reg .pred p<8>;\n\t.reg .f32 t<8>;\n\t"
        "setp.gt.s32 p0, %10, %11;\n\t"
        "setp.gt.s32 p1, %10, %11 + 1;\n\t"
        "setp.gt.s32 p2, %10, %11 + 2;\n\t"
        "setp.gt.s32 p3, %10, %11 + 3;\n\t"
        "setp.gt.s32 p4, %10, %11 + 4;\n\t"
        "setp.gt.s32 p5, %10, %11 + 5;\n\t"
        "setp.gt.s32 p6, %10, %11 + 6;\n\t"
        "setp.gt.s32 p7, %10, %11 + 7;\n\t"
        "@p0 ld.shared.f32 t0, [%0 + %12];\n\t"
        "@p1 ld.shared.f32 t1, [%0 + %12 + %13];\n\t"
        "@p2 ld.shared.f32 t2, [%0 + %12 + 2 * %13];\n\t"
        "@p3 ld.shared.f32 t3, [%0 + %12 + 3 * %13];\n\t"
        "@p4 ld.shared.f32 t4, [%0 + %12 + 4 * %13];\n\t"
        "@p5 ld.shared.f32 t5, [%0 + %12 + 5 * %13];\n\t"
        "@p6 ld.shared.f32 t6, [%0 + %12 + 6 * %13];\n\t"
        "@p7 ld.shared.f32 t7, [%0 + %12 + 7 * %13];\n\t"
        "@p0 fma.rn.f32 t0, %1, %9, t0;\n\t"
        "@p1 fma.rn.f32 t1, %2, %9, t1;\n\t"
        "@p2 fma.rn.f32 t2, %3, %9, t2;\n\t"
        "@p3 fma.rn.f32 t3, %4, %9, t3;\n\t"
        "@p4 fma.rn.f32 t4, %5, %9, t4;\n\t"
        "@p5 fma.rn.f32 t5, %6, %9, t5;\n\t"
        "@p6 fma.rn.f32 t6, %7, %9, t6;\n\t"
        "@p7 fma.rn.f32 t7, %8, %9, t7;\n\t"
        "@p0 st.shared.f32 [%0 + %12], t0;\n\t"
        "@p1 st.shared.f32 [%0 + %12 + %13], t1;\n\t"
        "@p2 st.shared.f32 [%0 + %12 + 2 * %13], t2;\n\t"
        "@p3 st.shared.f32 [%0 + %12 + 3 * %13], t3;\n\t"
        "@p4 st.shared.f32 [%0 + %12 + 4 * %13], t4;\n\t"
        "@p5 st.shared.f32 [%0 + %12 + 5 * %13], t5;\n\t"
        "@p6 st.shared.f32 [%0 + %12 + 6 * %13], t6;\n\t"
        "@p7 st.shared.f32 [%0 + %12 + 7 * %13], t7;\n\t}"
        ::"r"(addr), "f"(P[0]), "f"(P[1]), "f"(P[2]), "f"(P[3]), "f"(P[4]), "f"(P[5]), "f"(P[6]), "f"(P[7]), "f"(inv), "r"(len),
          "n"(J), "n"(IMM), "n"(STRIDE)
        : "memory");
}

// Unpredicated form of smem_fma_if8 (every lane owns all eight pixels).
template <int IMM, int STRIDE>
__device__ __forceinline__ void smem_fma8(uint32_t addr, const float* P, float inv) {
    asm volatile(
        "{\n\t.reg .f32 t<8>;\n\t"
        "ld.shared.f32 t0, [%0 + %10];\n\t"
        "ld.shared.f32 t1, [%0 + %10 + %11];\n\t"
        "ld.shared.f32 t2, [%0 + %10 + 2 * %11];\n\t"
        "ld.shared.f32 t3, [%0 + %10 + 3 * %11];\n\t"
        "ld.shared.f32 t4, [%0 + %10 + 4 * %11];\n\t"
        "ld.shared.f32 t5, [%0 + %10 + 5 * %11];\n\t"
        "ld.shared.f32 t6, [%0 + %10 + 6 * %11];\n\t"
        "ld.shared.f32 t7, [%0 + %10 + 7 * %11];\n\t"
        "fma.rn.f32 t0, %1, %9, t0;\n\t"
        "fma.rn.f32 t1, %2, %9, t1;\n\t"
        "fma.rn.f32 t2, %3, %9, t2;\n\t"
        "fma.rn.f32 t3, %4, %9, t3;\n\t"
        "fma.rn.f32 t4, %5, %9, t4;\n\t"
        "fma.rn.f32 t5, %6, %9, t5;\n\t"
        "fma.rn.f32 t6, %7, %9, t6;\n\t"
        "fma.rn.f32 t7, %8, %9, t7;\n\t"
        "st.shared.f32 [%0 + %10], t0;\n\t"
        "st.shared.f32 [%0 + %10 + %11], t1;\n\t"
        "st.shared.f32 [%0 + %10 + 2 * %11], t2;\n\t"
        "st.shared.f32 [%0 + %10 + 3 * %11], t3;\n\t"
        "st.shared.f32 [%0 + %10 + 4 * %11], t4;\n\t"
        "st.shared.f32 [%0 + %10 + 5 * %11], t5;\n\t"
        "st.shared.f32 [%0 + %10 + 6 * %11], t6;\n\t"
        "st.shared.f32 [%0 + %10 + 7 * %11], t7;\n\t}"
        ::"r"(addr), "f"(P[0]), "f"(P[1]), "f"(P[2]), "f"(P[3]), "f"(P[4]), "f"(P[5]), "f"(P[6]), "f"(P[7]), "f"(inv),
          "n"(IMM), "n"(STRIDE)
        : "memory");
}

// Pass 2: acc += P * inv over the same pixels (private region, one owner lane per pixel: plain read-modify-write).
template <int JB, int NJ, int HS, int BW, int NFULL = 0>
__device__ __forceinline__ void scatter_block(uint32_t aa, const float (&preg)[NJ], float inv, int len) {
    static_for<0, BW / 4>([&](auto kc) {
        constexpr int K = decltype(kc)::value, J = JB + 4 * K;
        if constexpr (NFULL == 8 && K == 0 && J + 7 < NJ) smem_fma8<4 * J * HS, 4 * HS>(aa, &preg[J], inv);
        else if constexpr (BW >= 8 && (K % 2 == 0) && J + 7 < NJ) smem_fma_if8<4 * J * HS, 4 * HS, J>(aa, &preg[J], inv, len);
        else if constexpr (BW >= 8 && (K % 2 == 1) && J + 3 < NJ) { /* second half of an eight */ }
        else if constexpr (J + 3 < NJ) smem_fma_if4<4 * J * HS, 4 * HS, J>(aa, preg[J], preg[J + 1], preg[J + 2], preg[J + 3], inv, len);
        else static_for<0, 4>([&](auto qc) {
            constexpr int Q = J + decltype(qc)::value;
            if constexpr (Q < NJ) smem_fma_if<4 * Q * HS, Q>(aa, preg[Q], inv, len);
        });
    });
}

template <int NJ, int HS, int BW>
__device__ __forceinline__ void piece_pass2(uint32_t aa, const float (&preg)[NJ], float inv, int len, int nblk, bool full8 = false) {
    constexpr int NB = (NJ + BW - 1) / BW;
#define JPET_SCATTER(B)                                                                      \
    do {                                                                                     \
        if ((B) == 0 && BW >= 8 && NJ >= 8 && full8) scatter_block<0, NJ, HS, BW, 8>(aa, preg, inv, len); \
        else scatter_block<(B) * BW, NJ, HS, BW>(aa, preg, inv, len);                        \
    } while (0)
    JPET_BLOCK_CASES(JPET_SCATTER)
#undef JPET_SCATTER
}

// Event records travel global -> shared with cp.async into a two-slot ring per warp, one event ahead: no registers
// are held across an event and the record is there when the warp comes back for it (an L1 prefetch hint was not:
// ncu showed 11 % of the samples waiting on the record's first use).
__device__ __forceinline__ void cp_async16(uint32_t saddr, const void* gptr) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(gptr) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ float4 lds128(uint32_t saddr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(saddr));
    return v;
}

__device__ __forceinline__ void named_barrier(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// One event on one group of NWE warps.  tab_n: table row of this event's row count ([lane of the group]).
template <int NWE, int NJA, int NJB, int HS, int DEG, int BW, bool VS>
__device__ __forceinline__ void process_event(const float4 r0, const float4 r1, const float4 r2, const float4 r3,
                                                    const DevParams& p, const uint32_t* tab_n, uint32_t w_addr, uint32_t a_addr,
                                                    int ry0, int rz0, int col_lo, int col_hi, float* red_s, int group, int glane,
                                                    int& my_evals, int& my_skipped, int& overflow) {
    constexpr int GL = NWE * 32;
    Piece A, B;
    pieces_setup<NJA, NJB, HS, DEG, VS>(tab_n[glane], r0, r1, r2, r3, p, ry0, rz0, col_lo, col_hi, A, B, overflow);
    const int nbA = (__reduce_max_sync(0xffffffffu, A.rc.len) + BW - 1) / BW;
    float pregA[NJA];
    // (one-warp groups only: in the 512-thread CTAs of the four-warp groups the second copy of block 0 costs more than it saves)
    const bool fullA = NWE == 1 && DEG > 0 && BW >= 8 && NJA >= 8 && __reduce_min_sync(0xffffffffu, A.rc.len) >= 8;
    float denom = piece_pass1<NJA, HS, DEG, BW, VS>(A, w_addr, p.pxs, nbA, pregA, fullA);
    my_evals += A.rc.len;
    constexpr int NJB1 = NJB > 0 ? NJB : 2;
    float pregB[NJB1];
    int nbB = 0;
    if constexpr (NJB > 0) {
        nbB = (__reduce_max_sync(0xffffffffu, B.rc.len) + BW - 1) / BW;
        denom += piece_pass1<NJB, HS, DEG, BW, VS>(B, w_addr, p.pxs, nbB, pregB);
        my_evals += B.rc.len;
    }
    // ---- denominator: sum over the group -----------------------------------------------------------------------
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) denom += __shfl_xor_sync(0xffffffffu, denom, d);
    if constexpr (NWE > 1) {
        if ((glane & 31) == 0) red_s[glane >> 5] = denom;
        named_barrier(1 + group, GL);
        denom = 0.f;
#pragma unroll
        for (int q = 0; q < NWE; ++q) denom += red_s[q];
    }
    const bool ok = (denom > 0.f) && (denom < 3.0e38f);
    if (!ok) { if (glane == 0) my_skipped += 1; return; }
    const float inv = 1.f / denom;
    piece_pass2<NJA, HS, BW>(a_addr + A.off, pregA, inv, A.rc.len, nbA, fullA);
    if constexpr (NJB > 0) piece_pass2<NJB, HS, BW>(a_addr + B.off, pregB, inv, B.rc.len, nbB);
}

// CTA = NG groups of NWE warps.  Work item = (sub-tile, chunk of sorted events): the CTA stages w once, group g
// takes events g, g + NG, ... of the chunk into its own accumulator region and flushes it with red.global.add.
template <int NWE, int NG, int NJA, int NJB, int HS, int MINB, int DEG, int BW, bool VS, bool CLS>
__global__ void __launch_bounds__(NWE * NG * 32, MINB)
mlem_rows_kernel(const EventRec* __restrict__ sorted, const WorkItem* __restrict__ items, int* __restrict__ meta,
                  const __grid_constant__ DevParams p, const float* __restrict__ wT, float* __restrict__ accT,
                  const uint32_t* __restrict__ tab, unsigned long long* __restrict__ counters, int cls) {
    pdl_wait();
    constexpr int GT = NWE * NG * 32, GL = NWE * 32;
    extern __shared__ __align__(16) float smem[];
    const int WZ = p.WZ, RS = HS * WZ;
    // Warp w of a CTA issues on scheduler w mod 4.  With four warps per event the k-th warp of every group would sit on
    // scheduler k: the four central warps (longest chords) of the four groups on one scheduler, the four cap warps on
    // another (ncu: issue-active 55 ... 70 % across the schedulers).  Rotating the roles by the group index gives every
    // scheduler one warp of each role (config 4, large_deg5: 26.2 -> 25.0 ms per 10^7 events).
    const int tid = threadIdx.x, group = tid / GL;
    const int glane = NWE == 4 ? ((((tid >> 5) + group) & 3) << 5) + (tid & 31) : tid - group * GL;
    float* w_s = smem;
    float* acc_s = smem + RS * (1 + group);
    uint32_t* tab_s = reinterpret_cast<uint32_t*>(smem + RS * (1 + NG));
    const uint32_t w_addr = (uint32_t)__cvta_generic_to_shared(w_s);
    const uint32_t a_addr = (uint32_t)__cvta_generic_to_shared(acc_s);
    __shared__ float red_s[NG][2][NWE];
    __shared__ int item_s[2];
    __shared__ __align__(16) float rec_s[NWE * NG][2][16];
    const int lane = tid & 31;
    const uint32_t rec_addr = (uint32_t)__cvta_generic_to_shared(&rec_s[tid >> 5][0][0]);
    const int n_tab = (p.nr_max - p.nr_min + 1) * GL;
    for (int i = tid; i < n_tab; i += GT) tab_s[i] = __ldg(tab + i);

    const int n_items = meta[kMetaItems];              // (CLS: the item range of the degree class is read per item)
    int my_evals = 0, my_skipped = 0, overflow = 0;
    unsigned long long tot_evals = 0;
    int parity = 0, ip = 0;

    while (true) {
        if (tid == 0) {
            if constexpr (CLS) {
                // next item of this launch's degree class: a run of the full items, then a run of the partly filled ones
                // (MetaWord, common.cuh); read from meta every time, nothing of it lives in registers across the event loop
                const int k = atomicAdd(meta + (cls ? kMetaCounter1 : kMetaCounter0), 1);
                const int n_full = meta[kMetaFull], f0 = meta[kMetaFull0], p0 = meta[kMetaPart0];
                const int seg1_lo = cls ? f0 : 0, seg1_n = cls ? n_full - f0 : f0;
                const int seg2_lo = n_full + (cls ? p0 : 0), seg2_n = cls ? meta[kMetaItems] - n_full - p0 : p0;
                item_s[ip] = k < seg1_n ? seg1_lo + k : (k < seg1_n + seg2_n ? seg2_lo + (k - seg1_n) : -1);
            } else {
                item_s[ip] = atomicAdd(meta + kMetaCounter0, 1);
            }
        }
        __syncthreads();                                   // also: every group is done with the previous w region
        const int item = item_s[ip];
        ip ^= 1;
        if (CLS ? item < 0 : item >= n_items) break;
        const WorkItem wi = items[item];
        const int bin = CLS && wi.bin >= p.nby * p.nbz ? wi.bin - p.nby * p.nbz : wi.bin;
        const int by = bin / p.nbz, bz = bin - by * p.nbz;
        const int ry0 = by * p.Sy - 2 * p.Hy, rz0 = bz * p.Sz - 2 * p.Hz;        // region origin (pixel indices)
        const int row_lo = max(0, ry0), row_hi = min(p.n_y - 1, ry0 + HS - 1);
        const int col_lo = max(0, rz0), col_hi = min(p.n_z - 1, rz0 + WZ - 1);
        const float4* rec = reinterpret_cast<const float4*>(sorted + wi.start);
        if (group < wi.count && lane < 4) cp_async16(rec_addr + 16 * lane, rec + 4 * group + lane);      // slot 0
        cp_async_commit();
        for (int i0 = tid; i0 < RS; i0 += 4 * GT) {        // stage w: several loads in flight per thread
            float v[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = i0 + q * GT;
                const int c = i / HS, r = i - c * HS;
                const int iz = rz0 + c, iy = ry0 + r;
                v[q] = 0.f;
                if (i < RS && iz >= col_lo && iz <= col_hi && iy >= row_lo && iy <= row_hi) v[q] = __ldg(wT + (size_t)iz * p.n_y + iy);
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int i = i0 + q * GT;
                if (i < RS) w_s[i] = v[q];
            }
        }
        for (int i = 4 * glane; i < RS; i += 4 * GL) *reinterpret_cast<float4*>(acc_s + i) = make_float4(0.f, 0.f, 0.f, 0.f);
        __syncthreads();
        uint32_t slot = 0;
        for (int q = group; q < wi.count; q += NG) {
            cp_async_wait_all();
            __syncwarp();
            const uint32_t ra = rec_addr + slot;
            const float4 r0 = lds128(ra), r1 = lds128(ra + 16), r2 = lds128(ra + 32), r3 = lds128(ra + 48);
            slot ^= 64u;
            if (q + NG < wi.count && lane < 4) cp_async16(rec_addr + slot + 16 * lane, rec + 4 * (q + NG) + lane);
            cp_async_commit();
            // the sort admitted the event to a regular bin because its row count is one the table holds (event_place);
            // the clamp keeps a corrupted record inside the table and reports it like an overflowing piece
            const int nrows = rows_count(__float_as_int(r3.w));
            const int tn = min(max(nrows - p.nr_min, 0), p.nr_max - p.nr_min);
            overflow |= tn != nrows - p.nr_min;
            const uint32_t* tab_n = tab_s + tn * GL;
            process_event<NWE, NJA, NJB, HS, DEG, BW, VS>(r0, r1, r2, r3, p, tab_n, w_addr, a_addr, ry0, rz0, col_lo, col_hi,
                                                   red_s[group][parity], group, glane, my_evals, my_skipped, overflow);
            parity ^= 1;
        }
        tot_evals += (unsigned long long)my_evals;
        my_evals = 0;
        if constexpr (NWE > 1) named_barrier(1 + group, GL); else __syncwarp();
        // flush the group's region into the global transposed accumulator
        for (int i = 4 * glane; i < RS; i += 4 * GL) {
            const float4 v = *reinterpret_cast<const float4*>(acc_s + i);
            const int c = i / HS, r = i - c * HS;
            const int iz = rz0 + c, iy = ry0 + r;
            if (iz < col_lo || iz > col_hi) continue;
            float* dst = accT + (size_t)iz * p.n_y + iy;
            if (v.x != 0.f && iy >= row_lo && iy <= row_hi) red_add_f32(dst, v.x);
            if (v.y != 0.f && iy + 1 >= row_lo && iy + 1 <= row_hi) red_add_f32(dst + 1, v.y);
            if (v.z != 0.f && iy + 2 >= row_lo && iy + 2 <= row_hi) red_add_f32(dst + 2, v.z);
            if (v.w != 0.f && iy + 3 >= row_lo && iy + 3 <= row_hi) red_add_f32(dst + 3, v.w);
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        tot_evals += __shfl_xor_sync(0xffffffffu, tot_evals, d);
        overflow |= __shfl_xor_sync(0xffffffffu, overflow, d);
    }
    if ((tid & 31) == 0 && tot_evals) atomicAdd(counters + 0, tot_evals);
    if (glane == 0 && my_skipped) atomicAdd(counters + 1, (unsigned long long)my_skipped);
    if ((tid & 31) == 0 && overflow) atomicAdd(counters + 2, 1ull);
}

}  // namespace jpet
