// design.hpp -- host-side float64 preparation of the SOS cascade for the blocked scan.
//
// Every section (b0 b1 b2 a0 a1 a2) of the stateful SOS IIR operator is
// rewritten as a 2-state linear system
//        s[n] = A s[n-1] + B x[n],      y[n] = C s[n-1] + D x[n]
// in one of two coordinate systems, chosen for fp32 conditioning:
//
//   KIND_T  transposed direct form II:  A = [[-a1, 1], [-a2, 0]],  B = (b1 - a1 b0, b2 - a2 b0),
//           C = (1, 0), D = b0.  5 FMA-class ops per sample.  Used when both poles are far
//           from z = +-1 (coefficient rounding then moves the response by < 1e-6).
//   KIND_R  normal ("coupled") form for a complex pole pair sigma +- i omega:
//           A = [[sigma, omega], [-omega, sigma]], B = (1, 0), C = (c1, c2), D = 1, with the
//           section's b0 factored out into one global gain.  6 ops per sample.  The state
//           coordinates are orthogonal, so rounding noise injected into the carried state is
//           not amplified by the long memory of poles next to z = 1.
//
// The blocked scan needs, per section: the fix-up rows C A^i (i < L), the block powers
// A^(len 2^d) for the warp-shuffle scan, and A^len / A^part for the carry-out.  All are computed
// here in float64 from the unrounded A and rounded to fp32 last.
#pragma once
#include <cmath>
#include <cstring>

namespace filark {

enum { KIND_T = 0, KIND_R = 1 };
constexpr int kSubBlock = 32;      // samples per lane in a full tile (L)
constexpr int kScanSteps = 5;      // log2(32 lanes)
constexpr double kUseNormalFormBelow = 0.05;   // |1 -+ p|^2 threshold, see DESIGN.md 4

struct Mat2 { double a, b, c, d; };             // [[a, b], [c, d]]
inline Mat2 mul(const Mat2& x, const Mat2& y) {
    return { x.a * y.a + x.b * y.c, x.a * y.b + x.b * y.d,
             x.c * y.a + x.d * y.c, x.c * y.b + x.d * y.d };
}
inline Mat2 ident() { return {1, 0, 0, 1}; }
inline Mat2 mpow(Mat2 m, long long e) {
    Mat2 r = ident();
    while (e > 0) { if (e & 1) r = mul(r, m); m = mul(m, m); e >>= 1; }
    return r;
}

struct Section {
    int kind;
    Mat2 A;
    double B[2], C[2], D;
    double gain;          // factor moved into the global input gain (1 for KIND_T)
    double coef[6];       // what the local pass multiplies with (meaning depends on kind)
    double pole_radius;
    double dist2;         // min(|1-p|^2, |1+p|^2)
};

enum DesignStatus { DESIGN_OK = 0, DESIGN_INVALID = 1, DESIGN_UNSTABLE = 2 };

// sos6: b0 b1 b2 a0 a1 a2
inline DesignStatus design_section(const double* sos6, Section* out)
{
    for (int i = 0; i < 6; ++i) if (!std::isfinite(sos6[i])) return DESIGN_INVALID;
    const double a0 = sos6[3];
    if (a0 == 0.0) return DESIGN_INVALID;
    const double b0 = sos6[0] / a0, b1 = sos6[1] / a0, b2 = sos6[2] / a0;
    const double a1 = sos6[4] / a0, a2 = sos6[5] / a0;
    // Jury conditions for both roots of z^2 + a1 z + a2 strictly inside the unit circle.
    if (!(std::fabs(a2) < 1.0 && std::fabs(a1) < 1.0 + a2)) return DESIGN_UNSTABLE;
    const double disc = a1 * a1 - 4.0 * a2;
    Section s{};
    s.dist2 = std::fmin(1.0 + a1 + a2, 1.0 - a1 + a2);
    s.gain = 1.0;
    if (disc < 0.0) s.pole_radius = std::sqrt(a2);
    else s.pole_radius = std::fmax(std::fabs((-a1 + std::sqrt(disc)) / 2), std::fabs((-a1 - std::sqrt(disc)) / 2));
    const double omega = disc < 0.0 ? 0.5 * std::sqrt(-disc) : 0.0;
    const bool normal_form = disc < 0.0 && b0 != 0.0 && omega > 1e-7 && s.dist2 < kUseNormalFormBelow;
    if (!normal_form) {
        s.kind = KIND_T;
        s.A = { -a1, 1.0, -a2, 0.0 };
        s.B[0] = b1 - a1 * b0; s.B[1] = b2 - a2 * b0;
        s.C[0] = 1.0; s.C[1] = 0.0; s.D = b0;
        s.coef[0] = b0; s.coef[1] = b1; s.coef[2] = b2; s.coef[3] = -a1; s.coef[4] = -a2; s.coef[5] = 0;
    } else {
        // Normalise the numerator by b0 (D = 1); b0 goes to the global gain.
        const double n1 = b1 / b0, n2 = b2 / b0;
        const double B1 = n1 - a1, B2 = n2 - a2;                 // DF2T input vector, D = 1
        const double sigma = -0.5 * a1;
        // T = [Re v, Im v], v = (1, -sigma + i omega): T^-1 A T = [[sigma, omega], [-omega, sigma]],
        // T^-1 B = (B1, (sigma B1 + B2)/omega), C T = (1, 0).
        const double Bp1 = B1, Bp2 = (sigma * B1 + B2) / omega;
        // M = [[Bp1, -Bp2], [Bp2, Bp1]] maps e1 -> B' and commutes with A': B'' = e1, C'' = C' M.
        s.kind = KIND_R;
        s.A = { sigma, omega, -omega, sigma };
        s.B[0] = 1.0; s.B[1] = 0.0;
        s.C[0] = Bp1; s.C[1] = -Bp2; s.D = 1.0;
        s.gain = b0;
        s.coef[0] = sigma; s.coef[1] = omega; s.coef[2] = s.C[0]; s.coef[3] = s.C[1];
        s.coef[4] = 0; s.coef[5] = 0;
    }
    *out = s;
    return DESIGN_OK;
}

// Fix-up rows g[i] = C A^i, i = 0 .. n-1 (out: 2n doubles, interleaved).
inline void fixup_rows(const Section& s, int n, double* out)
{
    double r0 = s.C[0], r1 = s.C[1];
    for (int i = 0; i < n; ++i) {
        out[2 * i] = r0; out[2 * i + 1] = r1;
        const double t0 = r0 * s.A.a + r1 * s.A.c, t1 = r0 * s.A.b + r1 * s.A.d;
        r0 = t0; r1 = t1;
    }
}

// Block powers for the scan over sub-blocks of `len` samples: P[d] = A^(len 2^d).
inline void scan_powers(const Section& s, int len, Mat2* P /* [kScanSteps] */)
{
    Mat2 m = mpow(s.A, len);
    for (int d = 0; d < kScanSteps; ++d) { P[d] = m; m = mul(m, m); }
}

}  // namespace filark
