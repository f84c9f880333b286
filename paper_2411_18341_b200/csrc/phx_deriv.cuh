// phx_deriv.cuh -- the derivative f of DESIGN.md section 2, step 1 (the paper's CALCULATE_K) for one cell of
// one component: five-point Laplacian Eq. (8); local terms of Eq. (1)/(16) PAPER.md:25, :361
// (sign and form as Listing 2); reservoir Eq. (17); compact nine-point TE-TM
// operator Delta_LT (d_x -+ i d_y)^2 on the other component.
// Used by the temporally blocked variants (STEP, RESIDENT).  Product code: shares nothing with oracle/.
#pragma once

#include "phx_common.cuh"

namespace phx {

// Nine-point neighbourhood of one component around a cell.  Scalar models read only c, w, e, s, n.
template <typename T>
struct Nbhd {
    typename Cx<T>::type c, w, e, s, n, sw, se, nw, ne;   // s = row j-1, n = row j+1, w = column i-1, e = column i+1
};

// K = i L - i W y + (Rr n / 2 - hgc) y - i J[other],  Kn = P - (gamr + Rr rho) n
//   own:    neighbourhood of this component (five-point part used)
//   oth:    neighbourhood of the other component (SPINOR only; all nine points used)
//   upper:  true for the psi_+ equation (operator (d_x - i d_y)^2 acts on psi_-)
template <typename T, bool SPINOR, bool RES>
__device__ __forceinline__ void deriv(const Coef<T>& k, const Nbhd<T>& own, const Nbhd<T>& oth, bool upper, T nres, T V, T P,
                                      T& Kr, T& Ki, T& Kn) {
    const auto y = own.c;
    const T rho = y.x * y.x + y.y * y.y - k.doff;
    // (hbar/2m) lap, Eq. (8)
    const T Lr = k.cx * (own.e.x + own.w.x - T(2) * y.x) + k.cy * (own.n.x + own.s.x - T(2) * y.x);
    const T Li = k.cx * (own.e.y + own.w.y - T(2) * y.y) + k.cy * (own.n.y + own.s.y - T(2) * y.y);
    T pot = V + k.g * rho;
    if (RES) pot += k.gr * nres;
    if (SPINOR) pot += k.gx * (oth.c.x * oth.c.x + oth.c.y * oth.c.y - k.doff);
    const T W = k.ih * pot;
    const T gain = RES ? (T(0.5) * k.Rr * nres - k.hgc) : -k.hgc;
    Kr = -Li + W * y.y + gain * y.x;
    Ki = Lr - W * y.x + gain * y.y;
    if (SPINOR) {
        const auto o = oth.c;
        const T dxx_r = oth.e.x + oth.w.x - T(2) * o.x, dxx_i = oth.e.y + oth.w.y - T(2) * o.y;
        const T dyy_r = oth.n.x + oth.s.x - T(2) * o.x, dyy_i = oth.n.y + oth.s.y - T(2) * o.y;
        const T dxy_r = oth.ne.x - oth.se.x - oth.nw.x + oth.sw.x, dxy_i = oth.ne.y - oth.se.y - oth.nw.y + oth.sw.y;
        const T sgn = upper ? T(-1) : T(1);
        const T Jr = k.bxx * dxx_r - k.byy * dyy_r - sgn * k.bxy * dxy_i;
        const T Ji = k.bxx * dxx_i - k.byy * dyy_i + sgn * k.bxy * dxy_r;
        Kr += Ji;
        Ki -= Jr;
    }
    Kn = RES ? P - (k.gamr + k.Rr * rho) * nres : T(0);
}

}  // namespace phx
