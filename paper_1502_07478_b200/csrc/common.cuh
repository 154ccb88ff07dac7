// common.cuh - shared device code of the list-mode MLEM hot path (sm_100a): the constants of a problem (DevParams),
// PTX wrappers, Eq. 2 per event, the 64-byte per-event record the sort writes, and the per-row form of Eq. 7 that
// the direct kernel and the evaluation counter use.
//
// Citations are /root/reference/PAPER.md lines.  Nothing here is shared with oracle/.
//
// Algebra (diagonal C^-1 = diag(iz2, iz2, il2), iz2 = 1/sigma_z^2, il2 = 1/sigma_dl^2; t = tan theta~,
// sec2 = 1 + t^2; pixel centre (y, z); dy = y - y~, dz = z - z~; u = dz - t dy; k = a3 coefficient).  With o, a, b of
// Eq. 8-10 written out, the four quadratic forms are
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
// sqrt(LH)), so P = r * ex2(c1s u^2 + c2s + (ba_s r)^2) with r = rsqrt(D).
// Row r of the ellipse is the closed interval |u| <= sqrt((9 - c2)/c1) (B.3 solved for dz), so pixels are
// enumerated by row spans and no lane is spent on a failed ellipse test (the paper's bbox + test wastes
// about one third of the lanes).
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
    // sigma_z as a function of the hit position: sigma_z(z) = sigma_z (1 + sz_eta min(1, z^2 inv_hL2)) (0 = constant)
    float sz_eta, inv_hL2, R;
    // binning and shared-memory regions (pixel units)
    int Hy, Hz;                        // halo on each side of a sub-tile
    int Sy, Sz;                        // sub-tile size
    int HS, WZ;                        // region: HS rows (y, fastest, multiple of 32) x WZ columns (z)
    int nby, nbz;                      // bins cover pixel indices [-Hy, n_y + Hy) x [-Hz, n_z + Hz)
    float t_max;                       // events with |tan theta~| above this go to the direct (global) path
    int chunk;                         // events per work item
    int nr_min, nr_max;                // ellipse row counts covered by the task table of the tiled event kernel;
                                       // nr_max > 0 makes the records carry the UNCLIPPED row range of the ellipse
    // degree classes (n_cls = 2): the sort puts the events whose OWN truncation bound allows the degree-3 exponent
    // polynomial (low_degree_ok) into a second set of bins, walked by the degree-3 instance of the kernel shape
    int n_cls;                         // 1: one class
    float cls_xk, cls_ylim, cls_tol;   // 2 u_max / 0.95 [mm], half image height [mm], bound in log2 units
};

// meta words of a sorted batch (BinSet::meta): the work-item list holds the full items (chunk events) of all bins in bin
// order, then the partly filled last items in bin order; the bins of degree class 0 come first.
enum MetaWord { kMetaItems = 0, kMetaDirectStart = 1, kMetaDirectCount = 2, kMetaCounter0 = 3, kMetaFull0 = 4, kMetaPart0 = 5,
                kMetaCounter1 = 6, kMetaFull = 7, kMetaWords = 8 };

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
// sigma_z of a strip as a function of the hit position ("depends on the z~u and z~d ... on the order of
// 10% from the center (lowest) to the edge (highest)"; reading R22): sigma_z(z) = sigma_z (1 + eta (2z/L)^2),
// |2z/L| clamped to 1.  eta = 0 is the paper's constant sigma_z.  Per event the inverse covariance becomes
// diag(iu, id, il2) (+ gamma), iu = 1/sigma_z(z~u)^2, id = 1/sigma_z(z~d)^2, and with S = iu + id, Dl = id - iu the
// forms of the header read
//   b.C^-1.b = S u^2 + 4 il2 sec2 dy^2          b.C^-1.a = -sec2 (S y + Dl R) u + 2 k il2 sec2 t y dy
//   a.C^-1.a = sec2^2 (S (y^2 + R^2) + 2 Dl R y) + k^2 il2 sec2 t^2 y^2
//   o.C^-1.b = -sec2 t (S y + Dl R) u + 2 il2 sec2 (1 + 2 t^2) y dy
// (b1 = b2, so the ellipse is the one of B.3 with 2 / sigma_z^2 replaced by S).
struct EventConsts {
    float t, sec2, y_t, z_t;
    float fy;           // y~ in pixel units (row index, fractional)
    float hy_px;        // half height of the ellipse in pixels
    float S, Dl;        // iu + id and id - iu [1/mm^2]  (2 / sigma_z^2 and 0 when sigma_z is constant)
    float inv_S;        // 1 / S
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
    e.S = p.d1k; e.Dl = 0.f; e.inv_S = p.half_sz2;
    if (p.sz_eta != 0.f) {
        const float qu = fminf(zu * zu * p.inv_hL2, 1.f), qd = fminf(zd * zd * p.inv_hL2, 1.f);
        const float su = fmaf(p.sz_eta, qu, 1.f), sd = fmaf(p.sz_eta, qd, 1.f);      // sigma_z(z) / sigma_z
        const float iu = 0.5f * p.d1k / (su * su), id = 0.5f * p.d1k / (sd * sd);
        e.S = iu + id; e.Dl = id - iu; e.inv_S = 1.f / e.S;
    }
    return e;
}

// Per-event form of the plan's truncation bound (jpet_api.cu make_plan) for the degree-3 exponent
// polynomial, gamma = 0 and constant sigma_z: with y_m the largest |y| the event's ellipse reaches inside the image,
//   x_e = 2 |t| / sec2 * y_m u_max / (R^2 + y_m^2) / 0.95,      e_e = 1.1 (3 y_m / sqrt(R^2 + y_m^2))^2,
// the neglected terms at the fraction s of the half chord are <= e_e (1 + x_e)^2 s^2 (x_e s)^2 / (2 (1 - x_e)) and
// (x_e s)^4 / 8, a kernel value there is <= 1.05 exp(-g s^2) of the event's peak, g = 4.5 (1 - e_e / 9), and
// max_s s^4 exp(-g s^2) = (2 / (g e))^2 for g > 2.  Evaluated in fp32 against 0.9 of the bound.
__device__ __forceinline__ bool low_degree_ok(const EventConsts& e, const DevParams& p) {
    const float ym = fminf(fabsf(e.y_t) + e.hy_px * p.px, p.cls_ylim);
    const float r2 = fmaf(ym, ym, p.R2);
    const float xe = p.cls_xk * fabsf(e.t) / e.sec2 * ym / r2;
    const float ee = 1.1f * 9.f * ym * ym / r2;
    const float g = 4.5f * (1.f - ee * (1.f / 9.f));
    if (!(g > 2.2f) || !(xe < 0.25f)) return false;
    const float m = 0.73575888f / g;                       // 2 / (g e)
    const float w = 1.05f * m * m;
    const float x2 = xe * xe, opx = 1.f + xe;
    const float err = 1.4427f * w * (0.5f * ee * opx * opx * x2 / (1.f - xe) + 0.125f * x2 * x2);
    return err <= 0.9f * p.cls_tol;
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
    float c1s;     // -LH * c1 (c1 = S)
    float c2s;     // -LH * c2
    float betas;   // sqrt(LH) * beta
    float delta;
    float alphas;  // sqrt(LH) * alpha
    float eps;
    int lo;        // first column of the row's span
    int len;       // pixels in the span
};

// Row constants and the span of row iy, clipped to columns [col_lo, col_hi].
__device__ __forceinline__ RowConsts row_setup(const EventConsts& e, int iy, int col_lo, int col_hi, const DevParams& p) {
    RowConsts r;
    float y = fmaf((float)iy, p.px, p.y0);
    float dy = y - e.y_t;
    float c2 = p.c2k * e.sec2 * dy * dy;
    float rem = 9.f - c2;                                  // row chord: c1 u^2 <= 9 - c2
    float hw = sqrt_approx(fmaxf(rem, 0.f) * e.inv_S);
    float zc = fmaf(e.t, dy, e.z_t);                       // u = 0 on the line z = z~ + t dy
    int lo = max(col_lo, __float2int_ru((zc - hw - p.z0) * p.inv_px));
    int hi = min(col_hi, __float2int_rd((zc + hw - p.z0) * p.inv_px));
    int len = rem >= 0.f ? max(0, hi - lo + 1) : 0;
    float alpha = -e.sec2 * fmaf(e.S, y, e.Dl * p.R);
    r.u0 = fmaf((float)lo, p.px, p.z0) - zc;
    r.c1s = -kLH * e.S;
    r.c2s = -kLH * c2;
    float ysec = y * e.sec2;
    r.betas = kSqrtLH * p.bk * ysec * e.t * dy;
    r.delta = e.sec2 * e.sec2 * fmaf(e.S, fmaf(y, y, p.R2), 2.f * e.Dl * p.R * y) + p.d2k * ysec * e.t * e.t * y
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

// P (up to the constant K) at pixel j of the row.
__device__ __forceinline__ float kernel_value(const RowConsts& r, float jf, float px) {
    float u = fmaf(jf, px, r.u0);
    float e2 = fmaf(r.c1s * u, u, r.c2s);
    float ba = fmaf(r.alphas, u, r.betas);
    float D = fmaf(r.eps, u, r.delta);
    float rs = rsqrt_approx(D);
    float bar = ba * rs;
    e2 = fmaf(bar, bar, e2);
    return rs * ex2_approx(e2);
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

// Per-event constants, written by bin_scatter_rec_kernel (sort_kernels.cuh), read (broadcast) by mlem_rows_kernel.
// Along the ellipse all row constants are polynomials in dy = y - y~ (y = y~ + dy):
//     c2s    = K2 dy^2                       betas = dy (B1 + KB dy)
//     alphas = A0 + A1 dy                    eps   = E0 + E1 dy
//     delta  = D0 + dy (D1 + D2 dy)
//     half chord^2 [pixels^2] = H0p / GS + H2p dy^2      chord centre [pixels] = Z0 + T1 dy
// u is rescaled with the constant-sigma_z factor sq (DevParams), so the Gaussian term along a row is -GS v^2 with
// GS = S / (2 / sigma_z^2): exactly 1 unless sigma_z depends on the hit positions.
struct __align__(16) EventRec {
    float yoff, K2, B1, KB;      // dy = iy * px + yoff;  c2s = K2 dy^2;  betas = dy (B1 + KB dy)
    float A0, A1, E0, E1;        // alphas = A0 + A1 dy;  eps = E0 + E1 dy
    float D0, D1, D2, H2p;       // delta = D0 + dy (D1 + D2 dy);  hw^2 = H0p / GS + H2p dy^2  (pixels^2)
    float Z0, T1;                // chord centre = Z0 + T1 dy  (pixels, column 0 = 0)
    float GS;                    // see above
    int rows;                    // (first row of the ellipse << 8) | number of rows (<= 255)
};
static_assert(sizeof(EventRec) == 64, "EventRec must be 64 bytes");

__device__ __forceinline__ int pack_rows(int iy_lo, int nrows) { return (int)(((unsigned)iy_lo << 8) | (unsigned)(nrows & 0xff)); }
__device__ __forceinline__ int rows_first(int rows) { return rows >> 8; }
__device__ __forceinline__ int rows_count(int rows) { return rows & 0xff; }

// Eq. 2 and the per-event factors of Eq. 7-10 / B.3 (see the header of this file for the algebra).
__device__ __forceinline__ EventRec make_event_rec(float zu, float zd, float dl, int rows, const DevParams& p) {
    const EventConsts e = event_setup(zu, zd, dl, p);
    EventRec r;
    const float t = e.t, sec2 = e.sec2, yt = e.y_t;
    const float s4 = sec2 * sec2, st2 = sec2 * t * t;
    r.yoff = p.y0 - yt;
    r.K2 = -kLH * p.c2k * sec2;
    r.KB = kSqrtLH * p.bk * sec2 * t;
    r.B1 = r.KB * yt;
    const float RD = e.Dl * p.R;                           // 0 for a constant sigma_z
    r.A1 = -kSqrtLH * e.S * sec2 * p.inv_sq;
    r.A0 = fmaf(r.A1, yt, -kSqrtLH * RD * sec2 * p.inv_sq);
    r.E1 = -2.f * t * e.S * sec2 * p.inv_sq;
    r.E0 = fmaf(r.E1, yt, -2.f * t * RD * sec2 * p.inv_sq);
    const float G1 = fmaf(p.d2k, st2, e.S * s4);
    const float G2 = p.d3k * fmaf(2.f, st2, sec2);
    r.D0 = fmaf(G1, yt * yt, e.S * s4 * p.R2) + 2.f * s4 * RD * yt;
    r.D1 = fmaf(fmaf(2.f, G1, G2), yt, 2.f * s4 * RD);
    r.D2 = G1 + G2;
    if (p.gB != 0.f) {                                     // Eq. 12 with gamma != 0 (DevParams)
        const float sec3 = sec2 * sec2 * rsqrt_approx(sec2);
        const float G3 = sec3 * t;
        r.B1 -= kSqrtLH * p.gB * sec3;
        r.D0 -= p.gD0 * G3 * yt;
        r.D1 -= (p.gD0 + 2.f * p.gB) * G3;
    }
    r.H2p = -p.c2k * sec2 * e.inv_S * p.inv_px * p.inv_px;
    r.Z0 = (e.z_t - p.z0) * p.inv_px;
    r.T1 = t * p.inv_px;
    r.GS = p.sz_eta != 0.f ? e.S * p.half_sz2 : 1.f;
    r.rows = rows;
    return r;
}

}  // namespace jpet
