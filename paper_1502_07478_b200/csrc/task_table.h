// task_table.h - host side: which piece of which ellipse row each lane of an event group walks (mlem_rows.cuh).
//
// The 3-sigma ellipse of an event (App. B :251-267) has half height hy = 1.5 sigma_dl cos(theta~)
// and, on the image row at signed distance d from its centre, a chord of half length sqrt(H0 (1 - (d/hy)^2)),
// H0 = 9 sigma_z^2 / 2, whatever the tilt (the tilt only shifts the chord).  In pixel units: for an ellipse
// that covers n rows, hy lies in [(n-1)/2, (n+1)/2] and row r (counted from the first covered row) sits at
// d in [r - hy, r - hy + 1); that bounds the number of pixel centres on row r from above by lenmax(n, r).
// The table assigns, for every n the plan can meet, the central 32*NWE rows whole to slot A (one row per lane,
// lane = row mod 32 inside its warp so that a warp's rows fall into distinct shared-memory banks) and the
// remaining cap rows to slot B, whole if lenmax fits the slot's capacity, else in 2 or 4 equal parts.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <vector>

namespace jpet_host {

constexpr uint32_t kTaskValid = 1u << 15;

inline uint32_t task_entry(int row, int part, int sh) { return kTaskValid | (uint32_t)row | ((uint32_t)part << 8) | ((uint32_t)sh << 10); }

// Upper bound of the pixel count of row r of an ellipse covering n rows; H0p = half chord^2 at the centre [px^2].
inline int row_len_max(int n, int r, double H0p) {
    double best = 0.0;
    const int steps = 64;
    for (int k = 0; k <= steps; ++k) {
        const double hy = std::max(0.25, 0.5 * (n - 1) + (double)k / steps);      // [(n-1)/2, (n+1)/2]
        const double lo = r - hy, hi = r - hy + 1.0;                                // d in [lo, hi)
        const double dmin = (lo <= 0.0 && hi >= 0.0) ? 0.0 : std::min(std::fabs(lo), std::fabs(hi));
        const double m = std::min(1.0, dmin / hy);
        best = std::max(best, H0p * (1.0 - m * m));
    }
    return (int)std::floor(2.0 * std::sqrt(best) + 1e-3) + 1;
}

// Builds the table [n - nr_min][lane], lanes = 32 * nwe: slot A in bits 0-15 of a word, slot B in bits 16-31.
// cap_b == 0: slot A only.  Returns false if some n in [nr_min, nr_max] does not fit the shape (too many rows, a
// chord longer than a slot).
inline bool build_task_table(int nr_min, int nr_max, double H0p, int nwe, int cap_a, int cap_b, std::vector<uint32_t>* out) {
    const int lanes = 32 * nwe;
    out->assign((size_t)(nr_max - nr_min + 1) * lanes, 0u);
    std::vector<uint32_t> A(lanes), B(lanes);
    for (int n = nr_min; n <= nr_max; ++n) {
        std::fill(A.begin(), A.end(), 0u);
        std::fill(B.begin(), B.end(), 0u);
        if (n > 255) return false;
        const int na = std::min(n, lanes);
        const int a0 = (n - na + 1) / 2;                       // central block [a0, a0 + na)
        // warp w of the group takes the rows at distance rank [32 w, 32 w + 32) from the block centre: 16 on either
        // side of the rows of warps 0..w-1 (warp 0: the central 32), so its chords are nearly equal
        const int c0 = a0 + (na - std::min(na, 32)) / 2;       // first row of the central 32
        for (int r = a0; r < a0 + na; ++r) {
            if (row_len_max(n, r, H0p) > cap_a) return false;
            int w, lane;
            if (r >= c0 && r < c0 + 32) { w = 0; lane = r - c0; }
            else if (r < c0) { const int k = c0 - 1 - r; w = 1 + k / 16; lane = 15 - (k % 16); }
            else { const int k = r - (c0 + 32); w = 1 + k / 16; lane = 16 + (k % 16); }
            if (w >= nwe) {                                     // uneven split of the block around the centre: use a free lane
                w = -1;
                for (int q = 0; q < lanes && w < 0; ++q)
                    if (A[q] == 0u) { w = q / 32; lane = q % 32; }
                if (w < 0) return false;
            }
            if (A[w * 32 + lane] != 0u) {
                int q = 0;
                while (q < lanes && A[q] != 0u) ++q;
                if (q == lanes) return false;
                w = q / 32; lane = q % 32;
            }
            A[w * 32 + lane] = task_entry(r, 0, 0);
        }
        if (n > na) {
            if (cap_b <= 0) return false;
            // cap rows, alternately below and above the block (longest first), whole or in 2 / 4 parts
            int next = 0;
            const int n_lo = a0, n_hi = n - (a0 + na);
            for (int k = 0; k < std::max(n_lo, n_hi); ++k) {
                for (int side = 0; side < 2; ++side) {
                    if (side == 0 && k >= n_lo) continue;
                    if (side == 1 && k >= n_hi) continue;
                    const int r = side == 0 ? a0 - 1 - k : a0 + na + k;
                    const int lm = row_len_max(n, r, H0p);
                    int sh = 0;
                    while (sh < 3 && (lm + (1 << sh) - 1) / (1 << sh) > cap_b) ++sh;
                    if (sh == 3) return false;
                    for (int part = 0; part < (1 << sh); ++part) {
                        if (next >= lanes) return false;
                        B[next++] = task_entry(r, part, sh);
                    }
                }
            }
        }
        uint32_t* W = out->data() + (size_t)(n - nr_min) * lanes;
        for (int q = 0; q < lanes; ++q) W[q] = A[q] | (B[q] << 16);
    }
    return true;
}

}  // namespace jpet_host
