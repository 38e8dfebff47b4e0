// design.hpp -- host-side float64 preparation of the SOS cascade for the blocked scan.
//
// Every section (b0 b1 b2 a0 a1 a2) of the stateful SOS IIR operator is
// rewritten as a 2-state linear system
//        s[n] = A s[n-1] + B x[n],      y[n] = C s[n-1] + D x[n]
// in a coordinate system chosen for fp32 conditioning and instruction count.
// With the numerator normalised to 1 + n1 z^-1 + n2 z^-2 (b0 moves into one global gain):
//
//   KIND_DF2    direct form II:  w = x - a1 w1 - a2 w2,  y = w + n1 w1 + n2 w2,  s = (w1, w2).
//               4 FMA per sample.  Used when both poles are far from z = +-1.
//   KIND_DF2G   the same with an explicit b0 (sections whose b0 is 0):  y = b0 w + b1 w1 + b2 w2.
//   KIND_DELTA  delta (difference) form for poles next to z = +1, s = (u, w), u = w[n] - w[n-1]:
//                    u' = p u - q w + x,   w' = w + u',   y = u' - n2 u  (+ m w),
//               p = a2, q = 1 + a1 + a2, m = 1 + n1 + n2.  The large, slowly varying state w is
//               only ever multiplied by the tiny q, and q = |1 - pole|^2 keeps full relative
//               precision in fp32 -- the two things direct forms lose next to z = 1.
//               4 FMA per sample when the section has a zero at z = 1 (m = 0), else 5
//               (KIND_DELTAG).
//   KIND_NORMAL normal ("coupled") form for a complex pole pair sigma +- i omega next to
//               z = -1:  A = [[sigma, omega], [-omega, sigma]], B = e1, C = (c1, c2), D = 1.
//               6 FMA per sample.
//
// The blocked scan needs, per section and per sub-block length L: the fix-up rows C A^i (i < L),
// the powers A^r (r <= L) for the carry across a (possibly short) sub-block, and A^(2L 2^d) for
// the warp-shuffle scan over lane pairs.  All are computed here in float64 from the unrounded A
// and rounded to fp32 last.
#pragma once
#include <cmath>
#include <cstring>

namespace filark {

enum { KIND_DF2 = 0, KIND_DF2G = 1, KIND_DELTA = 2, KIND_DELTAG = 3, KIND_NORMAL = 4 };
constexpr double kNearUnitCircle = 0.05;   // |1 -+ pole|^2 threshold, see DESIGN.md 4

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
inline double norm1(const Mat2& m) {
    return std::fmax(std::fabs(m.a) + std::fabs(m.c), std::fabs(m.b) + std::fabs(m.d));
}

struct Section {
    int kind;
    Mat2 A;
    double B[2], C[2], D;
    double gain;          // factor moved into the global input gain (1 for KIND_DF2G)
    double coef[6];       // what the local pass multiplies with (meaning depends on kind)
    double pole_radius;
    double dist_p1, dist_m1;     // |1 - p|^2 = 1 + a1 + a2,  |1 + p|^2 = 1 - a1 + a2
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
    s.dist_p1 = 1.0 + a1 + a2;
    s.dist_m1 = 1.0 - a1 + a2;
    s.gain = 1.0;
    if (disc < 0.0) s.pole_radius = std::sqrt(a2);
    else s.pole_radius = std::fmax(std::fabs((-a1 + std::sqrt(disc)) / 2), std::fabs((-a1 - std::sqrt(disc)) / 2));
    const double omega = disc < 0.0 ? 0.5 * std::sqrt(-disc) : 0.0;
    if (b0 == 0.0) {
        s.kind = KIND_DF2G;
        s.A = { -a1, -a2, 1.0, 0.0 };
        s.B[0] = 1.0; s.B[1] = 0.0;
        s.C[0] = b1; s.C[1] = b2; s.D = 0.0;
        s.coef[0] = -a1; s.coef[1] = -a2; s.coef[2] = b1; s.coef[3] = b2; s.coef[4] = 0.0;
        *out = s;
        return DESIGN_OK;
    }
    const double n1 = b1 / b0, n2 = b2 / b0;       // numerator 1 + n1 z^-1 + n2 z^-2, gain b0
    s.gain = b0;
    s.D = 1.0;
    if (s.dist_p1 < kNearUnitCircle) {
        const double p = a2, q = s.dist_p1;
        double m = 1.0 + n1 + n2;
        if (std::fabs(m) < 1e-13 * (1.0 + std::fabs(n1) + std::fabs(n2))) m = 0.0;   // zero at z = 1
        s.kind = m == 0.0 ? KIND_DELTA : KIND_DELTAG;
        s.A = { p, -q, p, 1.0 - q };
        s.B[0] = 1.0; s.B[1] = 1.0;
        s.C[0] = p - n2; s.C[1] = m - q;
        s.coef[0] = p; s.coef[1] = -q; s.coef[2] = -n2; s.coef[3] = m; s.coef[4] = p - q;
    } else if (s.dist_m1 < kNearUnitCircle && disc < 0.0 && omega > 1e-7) {
        const double B1 = n1 - a1, B2 = n2 - a2;                 // DF2T input vector, D = 1
        const double sigma = -0.5 * a1;
        // T = [Re v, Im v], v = (1, -sigma + i omega): T^-1 A T = [[sigma, omega], [-omega, sigma]],
        // T^-1 B = (B1, (sigma B1 + B2)/omega), C T = (1, 0).  M = [[Bp1, -Bp2], [Bp2, Bp1]] maps
        // e1 -> B' and commutes with A': B'' = e1, C'' = C' M.
        const double Bp1 = B1, Bp2 = (sigma * B1 + B2) / omega;
        s.kind = KIND_NORMAL;
        s.A = { sigma, omega, -omega, sigma };
        s.B[0] = 1.0; s.B[1] = 0.0;
        s.C[0] = Bp1; s.C[1] = -Bp2;
        s.coef[0] = sigma; s.coef[1] = omega; s.coef[2] = s.C[0]; s.coef[3] = s.C[1];
    } else {
        s.kind = KIND_DF2;
        s.A = { -a1, -a2, 1.0, 0.0 };
        s.B[0] = 1.0; s.B[1] = 0.0;
        s.C[0] = n1 - a1; s.C[1] = n2 - a2;
        s.coef[0] = -a1; s.coef[1] = -a2; s.coef[2] = n1; s.coef[3] = n2;
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

// 1 - (1-c)^e, accurate for tiny c (the averages' block decay in the "v += u - beta u" form).
inline double one_minus_pow(double c, double e)
{
    if (e <= 0.0) return 0.0;
    if (c >= 1.0) return 1.0;
    return -std::expm1(e * std::log1p(-c));
}

}  // namespace filark
