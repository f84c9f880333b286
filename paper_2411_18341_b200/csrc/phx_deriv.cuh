// phx_deriv.cuh -- the derivative f of DESIGN.md section 2, step 1 (the paper's CALCULATE_K) for one cell of
// one component: five-point Laplacian Eq. (8); local terms of Eq. (1)/(16) PAPER.md:25, :361
// (sign and form as Listing 2); reservoir Eq. (17); compact nine-point TE-TM
// operator Delta_LT (d_x -+ i d_y)^2 on the other component.
// Used by the temporally blocked variant STEP.  Product code: shares nothing with oracle/.
//
// Written on (re, im) PAIRS: for complex fp32 every pair operation below is one packed sm_100 instruction
// (FADD2 / FMUL2 / FFMA2 on a 64-bit register pair), and multiplication by +-i is an operand modifier of that
// instruction (swap + one-sided negation), not an instruction.  The pair ops have the same flop throughput as the
// scalar ones but take half the issue slots, which is what bounds variant STEP (DESIGN.md sections 5.2 and 6).
// For complex fp64 the same code expands to scalar DADD/DMUL/DFMA.
#pragma once

#include "phx_common.cuh"

namespace phx {

// ---- pair arithmetic -------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2s(float s, float2 a) { return __fmul2_rn(make_float2(s, s), a); }
__device__ __forceinline__ float2 fma2s(float s, float2 a, float2 c) { return __ffma2_rn(make_float2(s, s), a, c); }   // s*a + c

__device__ __forceinline__ double2 add2(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 sub2(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ double2 fma2(double2 a, double2 b, double2 c) { return make_double2(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)); }
__device__ __forceinline__ double2 mul2s(double s, double2 a) { return make_double2(s * a.x, s * a.y); }
__device__ __forceinline__ double2 fma2s(double s, double2 a, double2 c) { return make_double2(fma(s, a.x, c.x), fma(s, a.y, c.y)); }

// i*a (a free operand modifier of the packed instructions when it is the addend)
__device__ __forceinline__ float2 rot(float2 a) { return make_float2(-a.y, a.x); }
__device__ __forceinline__ double2 rot(double2 a) { return make_double2(-a.y, a.x); }

// Neighbourhood of one component around a cell: the five points of Eq. (8) and, for the TE-TM operator, the
// undivided corner difference D = Dxy4 = (n - s)[east column] - (n - s)[west column] (set by the spinor models only).
template <typename T>
struct Nbhd {
    typename Cx<T>::type c, w, e, s, n, D;   // s = row j-1, n = row j+1, w = column i-1, e = column i+1
};

// Differences of one component at a cell: L = (hbar/2m) lap, Eq. (8); for the TE-TM operator also the undivided
// A = Dxx, B = Dyy and D = Dxy4 (corners).
template <typename T>
struct Diff {
    typename Cx<T>::type L, A, B, D;
};

// NINE: the spinor models (all nine points, A, B, D kept).  ISO: dx == dy, so cx == cy and
// L = cx ((e + w) + (n + s) - 4 c) -- one packed operation fewer, exact factors only.  NINE and ISO: bxx == byy as well
// (both are beta / (hbar d^2) of the same d), so the TE-TM operator needs only A - B = (e + w) - (n + s), kept in A.
template <typename T, bool NINE, bool ISO>
__device__ __forceinline__ void differences(const Coef<T>& k, const Nbhd<T>& nb, Diff<T>& d) {
    if (ISO && !NINE) {
        d.L = mul2s(k.cx, fma2s(T(-4), nb.c, add2(add2(nb.e, nb.w), add2(nb.n, nb.s))));
    } else if (ISO) {
        const typename Cx<T>::type ew = add2(nb.e, nb.w), ns = add2(nb.n, nb.s);
        d.L = mul2s(k.cx, fma2s(T(-4), nb.c, add2(ew, ns)));
        d.A = sub2(ew, ns);
    } else {
        d.A = fma2s(T(-2), nb.c, add2(nb.e, nb.w));
        d.B = fma2s(T(-2), nb.c, add2(nb.n, nb.s));
        d.L = fma2s(k.cy, d.B, mul2s(k.cx, d.A));
    }
    if (NINE) d.D = nb.D;
}

// K = i L - i W y + (Rr n / 2 - hgc) y - i J[other],  Kn = P - (gamr + Rr rho) n
//   y, own:  this component's value and differences;  yo, oth: the other component's (SPINOR only)
//   upper:   true for the psi_+ equation (operator (d_x - i d_y)^2 acts on psi_-)
//   Ed, q:  drive amplitude E(r) of the cell and q = (1/hbar) exp(-i omega t_s) (DRIVE only):  K += -i q E
//   UNITH:  ih == 1 exactly (units with hbar = 1, as Eq. (1) is benchmarked: BASELINE configs 1, 2, 4): the product ih * pot is
//           pot itself, bit for bit, and its multiplication is not issued
template <typename T, bool SPINOR, bool RES, bool DRIVE, bool ISO = false, bool UNITH = false>
__device__ __forceinline__ typename Cx<T>::type deriv(const Coef<T>& k, typename Cx<T>::type y, const Diff<T>& own,
                                                      typename Cx<T>::type yo, const Diff<T>& oth, bool upper, T nres, T V,
                                                      T P, typename Cx<T>::type Ed, typename Cx<T>::type q, T& Kn) {
    using C = typename Cx<T>::type;
    const T rho = fma(y.y, y.y, fma(y.x, y.x, -k.doff));
    T pot = fma(k.g, rho, V);
    if (RES) pot = fma(k.gr, nres, pot);
    if (SPINOR) pot = fma(k.gx, fma(yo.y, yo.y, fma(yo.x, yo.x, -k.doff)), pot);
    const T W = UNITH ? pot : k.ih * pot;
    const T gain = RES ? fma(T(0.5) * k.Rr, nres, -k.hgc) : -k.hgc;
    // K = i M + gain y -+ bxy Dxy4[other],  M = L - W y - bxx Dxx[other] + byy Dyy[other]
    // (-i J with J = bxx Dxx - byy Dyy -+ i bxy Dxy4 of the other component; the one rotation sits on the addend
    // operand, where the packed instruction takes it as a modifier)
    C M = fma2s(-W, y, own.L);
    if (SPINOR) {
        M = fma2s(-k.bxx, oth.A, M);                 // (ISO: oth.A holds Dxx - Dyy and bxx == byy)
        if (!ISO) M = fma2s(k.byy, oth.B, M);
    }
    // -i q E = i (-q_re E) + q_im E: the first part joins M (rotated below), the second K
    if (DRIVE) M = fma2s(-q.x, Ed, M);
    C K = fma2s(gain, y, rot(M));
    if (DRIVE) K = fma2s(q.y, Ed, K);
    if (SPINOR) K = fma2s(upper ? -k.bxy : k.bxy, oth.D, K);
    Kn = RES ? P - (k.gamr + k.Rr * rho) * nres : T(0);
    return K;
}

}  // namespace phx
