// generator.cuh - event simulation on the device: phantom sampling, acceptance by the two strips,
// Gaussian smearing - the recipe of DESIGN.md section 5 ("simulated data using realistic parameters", PAPER.md:204;
// phantom rule "topmost row wins"; forward model Eq. 1).
//
// Every event slot has its own counter-based random stream, Philox4x32-10 with key = (seed low, seed high) and counter
// = (slot low, slot high, attempt, block): block 0 gives the four uniforms of attempt `attempt` (y, z, acceptance,
// theta), block 1 the four uniforms of the Box-Muller smearing of the accepted attempt.  A 32-bit word x becomes the
// uniform ((x >> 8) + 0.5) 2^-24 in (0, 1), exactly representable in fp32.  Slot i is therefore the same event whatever
// the launch shape; the oracle implements the same generator in fp64 (same words, same decisions up to rounding at a
// boundary).
#pragma once
#include "common.cuh"

namespace jpet {

constexpr int kMaxPrimitives = 16;
constexpr int kMaxAttempts = 1 << 16;

struct PhantomDev {
    int n;
    int kind[kMaxPrimitives];                                              // 0 = ellipse, 1 = box
    float cy[kMaxPrimitives], cz[kMaxPrimitives], inv_hy[kMaxPrimitives], inv_hz[kMaxPrimitives];
    float cphi[kMaxPrimitives], sphi[kMaxPrimitives], rel[kMaxPrimitives];  // rel = intensity / max intensity
    float y0, y1, z0, z1;                                                   // bounding rectangle
    float R, half_L, sigma_z, sigma_dl;
};

struct Philox4 { uint32_t v[4]; };

__host__ __device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1) {
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)M0 * c0, p1 = (unsigned long long)M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    Philox4 o;
    o.v[0] = c0; o.v[1] = c1; o.v[2] = c2; o.v[3] = c3;
    return o;
}

__device__ __forceinline__ float uniform24(uint32_t x) { return ((float)(x >> 8) + 0.5f) * 5.9604644775390625e-8f; }

// Relative intensity at (y, z): the first primitive of the list that contains the point, 0 outside all.
__device__ __forceinline__ float phantom_rel(const PhantomDev& ph, float y, float z) {
    for (int k = 0; k < ph.n; ++k) {
        const float dz = z - ph.cz[k], dy = y - ph.cy[k];
        const float a = (ph.cphi[k] * dz + ph.sphi[k] * dy) * ph.inv_hz[k], b = (ph.cphi[k] * dy - ph.sphi[k] * dz) * ph.inv_hy[k];
        const bool in = ph.kind[k] == 0 ? (a * a + b * b <= 1.f) : (fabsf(a) <= 1.f && fabsf(b) <= 1.f);
        if (in) return ph.rel[k];
    }
    return 0.f;
}

__global__ void __launch_bounds__(256)
generate_events_kernel(float* __restrict__ events, long long n, unsigned long long first, unsigned long long seed,
                       const __grid_constant__ PhantomDev ph) {
    const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const unsigned long long slot = first + (unsigned long long)i;
        const uint32_t s0 = (uint32_t)slot, s1 = (uint32_t)(slot >> 32);
        float zu = __int_as_float(0x7fc00000), zd = zu, dl = zu;          // NaN if no attempt is accepted (skipped by MLEM)
        for (int a = 0; a < kMaxAttempts; ++a) {
            const Philox4 u = philox4x32_10(s0, s1, (uint32_t)a, 0u, k0, k1);
            const float y = fmaf(ph.y1 - ph.y0, uniform24(u.v[0]), ph.y0), z = fmaf(ph.z1 - ph.z0, uniform24(u.v[1]), ph.z0);
            if (!(uniform24(u.v[2]) < phantom_rel(ph, y, z))) continue;
            const float theta = 3.14159265358979f * (uniform24(u.v[3]) - 0.5f);
            float st, ct;
            sincosf(theta, &st, &ct);
            const float tt = st / ct;
            const float hu = fmaf(ph.R - y, tt, z), hd = fmaf(-(ph.R + y), tt, z);                 // hit points (Fig. 1)
            if (!(fabsf(hu) <= ph.half_L && fabsf(hd) <= ph.half_L)) continue;
            const Philox4 g = philox4x32_10(s0, s1, (uint32_t)a, 1u, k0, k1);
            const float r0 = sqrtf(-2.f * logf(uniform24(g.v[0]))), r1 = sqrtf(-2.f * logf(uniform24(g.v[2])));
            float s_a, c_a, s_b, c_b;
            sincosf(6.28318530717959f * uniform24(g.v[1]), &s_a, &c_a);
            sincosf(6.28318530717959f * uniform24(g.v[3]), &s_b, &c_b);
            (void)s_b;
            zu = fmaf(ph.sigma_z, r0 * c_a, hu);
            zd = fmaf(ph.sigma_z, r0 * s_a, hd);
            dl = fmaf(ph.sigma_dl, r1 * c_b, -2.f * y / ct);                                         // Eq. 1 on the LOR
            break;
        }
        events[3 * i] = zu;
        events[3 * i + 1] = zd;
        events[3 * i + 2] = dl;
    }
}

}  // namespace jpet
