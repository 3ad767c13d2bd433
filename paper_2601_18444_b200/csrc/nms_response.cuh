// nms_response.cuh -- pointwise response functions of Section II (L35-L174) from the four complex
// amplitudes, in fp64, in the two-component ("T") form of the Halpern-Johnson vector.
//
// With q^ = (0, s, c), s = sin th, c = cos th (Eq. 6), Eq. 7 (L62) gives
//     Q = q^ x (q^ x M) = (-Mx, -My c^2 + Mz s c, My s c - Mz s^2) = (-Mx, c T, -s T),  T = s Mz - c My,
// so |Q|^2 = |Mx|^2 + |T|^2 (Eq. 4), Pi = P.Q = -Px Mx + (Py c - Pz s) T (Eq. 8), and
// -i P.(Q x Q*) = 2 (Py s + Pz c) Im(T Mx*) (Eq. 14; the x component of Q x Q* vanishes identically,
// which is the "chi = 0 for P || e_x" of L100).  The remaining kinds are the sums of Eq. 11-13,
// 16-18, 23-24, 27.  (The oracle codes the same quantities from the cross-product definition.)
#pragma once
#include "../../include/nms.h"

namespace nms {

struct RespParams {
    double Px, Py, Pz;   // unit polarisation
    double sN, sM, invV; // DESIGN.md reading 4
};

// A[8] = Re N, Im N, Re Mx, Im Mx, Re My, Im My, Re Mz, Im Mz (raw sums); val[NMS_KIND_COUNT].
__device__ __forceinline__ void responses_at_point(const double A[8], double s, double c, const RespParams& p,
                                                   double val[NMS_KIND_COUNT])
{
    const double nr = p.sN * A[0], ni = p.sN * A[1];
    const double xr = p.sM * A[2], xi = p.sM * A[3];
    const double yr = p.sM * A[4], yi = p.sM * A[5];
    const double zr = p.sM * A[6], zi = p.sM * A[7];
    const double tr = s * zr - c * yr, ti = s * zi - c * yi;          // T
    const double g = p.Py * c - p.Pz * s;
    const double pr = -p.Px * xr + g * tr, pi = -p.Px * xi + g * ti;   // Pi = P.Q
    const double nuc = nr * nr + ni * ni;                              // Eq. 3
    const double mag = xr * xr + xi * xi + tr * tr + ti * ti;          // Eq. 4
    const double proj = pr * pr + pi * pi;                             // Eq. 8
    const double nm = 2.0 * (nr * pr + ni * pi);                       // Eq. 18: N Pi* + N* Pi
    const double chi = 2.0 * (p.Py * s + p.Pz * c) * (ti * xr - tr * xi);   // Eq. 14: Im(T Mx*)
    const double sf = mag - proj;                                      // Eq. 13
    const double pm = sf + chi, mp = sf - chi;                         // Eq. 11-12
    const double pp = nuc + nm + proj, mm = nuc - nm + proj;           // Eq. 16-17
    val[NMS_NUC] = p.invV * nuc;
    val[NMS_MAG] = p.invV * mag;
    val[NMS_UNPOL] = p.invV * (nuc + mag);                             // Eq. 27-28
    val[NMS_PROJ] = p.invV * proj;
    val[NMS_NM] = p.invV * nm;
    val[NMS_SF] = p.invV * sf;
    val[NMS_CHI] = p.invV * chi;
    val[NMS_PM] = p.invV * pm;
    val[NMS_MP] = p.invV * mp;
    val[NMS_PP] = p.invV * pp;
    val[NMS_MM] = p.invV * mm;
    val[NMS_POL_PLUS] = p.invV * (pp + pm);                            // Eq. 23
    val[NMS_POL_MINUS] = p.invV * (mm + mp);                           // Eq. 24
}

}  // namespace nms
