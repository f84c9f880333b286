// phx_stage.cuh -- variant STAGE: one fused kernel per Runge-Kutta stage.
//
// Per stage s the kernel reads the stage input y_s with a one-cell halo, evaluates the derivative
// (five-point Laplacian Eq. (8); local terms of Eq. (1)/(16) PAPER.md:25,:361; reservoir
// Eq. (17); TE-TM nine-point operator PAPER.md:367), and in the same pass writes the next
// stage input y_{s+1} = psi + a_s dt K_s (Eqs. (3)-(5)) and the running sum of Eq. (6); K_s never
// reaches memory.  Stage 4 writes psi(t+dt) and adds the Wiener increment of Eq. (22).
//
// Thread mapping: a thread owns VEC consecutive cells in x (one 128-bit load of complex fp32 pairs /
// one complex fp64) and walks `rows` rows in y with a register sliding window (rows j-1, j, j+1, and
// j+2 in flight), so every stage-input row is loaded once per CTA.  x neighbours come from warp
// shuffles; only the two edge lanes of a warp issue an extra (L1/L2-hit) load.  Periodic wrap and zero
// boundaries are resolved in the index computation.
#pragma once

#include "phx_common.cuh"
#include "phx_philox.cuh"

// Rows the DRAM -> L2 prefetch of the per-stage kernels runs ahead of the register prefetch (0 = none).  Same-run A/B at
// 4 rows (Gcell*step/s): cfg2 4096^2 fp32 43.0 against 40.2 (84 % of the measured HBM bandwidth on the 128 algorithmic bytes),
// cfg3 30.6 against 29.7, the 16384^2 spinor 20.2 against 21.0 (it has enough bytes in flight already); 8 rows lose everywhere,
// and so do 4 on an L2-resident grid (1024^2 fp32 27.0 against 29.7): Geom::pf switches it on for working sets beyond L2.
#ifndef PHX_STAGE_PF_ROWS
#define PHX_STAGE_PF_ROWS 4
#endif
#ifndef PHX_STAGE_PF_ROWS_SPINOR
#define PHX_STAGE_PF_ROWS_SPINOR 0
#endif
#ifndef PHX_STAGE_PF_ROWS_SPINOR1
#define PHX_STAGE_PF_ROWS_SPINOR1 0     // (stage 1 of the spinor models, the one with the fewest bytes in flight)
#endif

namespace phx {

template <typename T>
struct StageArgs {
    Geom geo;
    Coef<T> k;
    Fields<T> f;
    uint32_t seed;
};

template <typename T, int VEC>
struct Row {
    typename Cx<T>::type c[VEC];   // the thread's own cells
    typename Cx<T>::type el, er;   // x-1 / x+VEC, fetched from memory by warp-edge lanes only
};

// ---- vector loads / stores of VEC complex or real values -------------------------------------
template <int VEC> __device__ __forceinline__ void ld_c(const float2* p, float2 (&v)[VEC]) {
    if constexpr (VEC == 2) { const float4 q = *reinterpret_cast<const float4*>(p); v[0] = make_float2(q.x, q.y); v[1] = make_float2(q.z, q.w); }
    else { v[0] = *p; }
}
template <int VEC> __device__ __forceinline__ void ld_c(const double2* p, double2 (&v)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) v[i] = p[i];
}
template <int VEC> __device__ __forceinline__ void st_c(float2* p, const float2 (&v)[VEC]) {
    if constexpr (VEC == 2) *reinterpret_cast<float4*>(p) = make_float4(v[0].x, v[0].y, v[1].x, v[1].y);
    else *p = v[0];
}
template <int VEC> __device__ __forceinline__ void st_c(double2* p, const double2 (&v)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) p[i] = v[i];
}
template <int VEC> __device__ __forceinline__ void ld_r(const float* p, float (&v)[VEC]) {
    if constexpr (VEC == 2) { const float2 q = *reinterpret_cast<const float2*>(p); v[0] = q.x; v[1] = q.y; }
    else { v[0] = *p; }
}
template <int VEC> __device__ __forceinline__ void ld_r(const double* p, double (&v)[VEC]) {
    if constexpr (VEC == 2) { const double2 q = *reinterpret_cast<const double2*>(p); v[0] = q.x; v[1] = q.y; }
    else { v[0] = *p; }
}
template <int VEC> __device__ __forceinline__ void st_r(float* p, const float (&v)[VEC]) {
    if constexpr (VEC == 2) *reinterpret_cast<float2*>(p) = make_float2(v[0], v[1]);
    else *p = v[0];
}
template <int VEC> __device__ __forceinline__ void st_r(double* p, const double (&v)[VEC]) {
    if constexpr (VEC == 2) *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
    else *p = v[0];
}

__device__ __forceinline__ float2 shfl_up1(float2 v) { return make_float2(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ float2 shfl_dn1(float2 v) { return make_float2(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ double2 shfl_up1(double2 v) { return make_double2(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ double2 shfl_dn1(double2 v) { return make_double2(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1)); }

// Per-thread column bookkeeping: where the x neighbours of the thread's cells come from.
struct Cols {
    int x0;                 // first owned cell
    int xl, xr;             // wrapped neighbour columns
    bool active;            // x0 < nx
    bool l_shfl, r_shfl;    // neighbour is held by lane-1 / lane+1
    bool l_load, r_load;    // neighbour must be fetched from memory (warp edge)
};

template <int VEC>
__device__ __forceinline__ Cols make_cols(const Geom& g) {
    Cols c;
    const int lane = threadIdx.x & 31;
    c.x0 = (blockIdx.x * blockDim.x + threadIdx.x) * VEC;
    c.active = c.x0 < g.nx;
    c.xl = c.x0 - 1;
    c.xr = c.x0 + VEC;
    bool l_ok = true, r_ok = true;
    if (c.xl < 0) { if (g.bc_x) l_ok = false; else c.xl += g.nx; }
    if (c.xr >= g.nx) { if (g.bc_x) r_ok = false; else c.xr -= g.nx; }
    c.l_shfl = lane > 0;
    c.r_shfl = lane < 31 && (c.x0 + VEC) < g.nx;
    c.l_load = c.active && !c.l_shfl && l_ok;
    c.r_load = c.active && !c.r_shfl && r_ok;
    return c;
}

// Load row j (may be -1 or ny: wrapped or zero) of a complex plane.
template <typename T, int VEC>
__device__ __forceinline__ void load_row(const typename Cx<T>::type* plane, int j, const Geom& g, const Cols& c, Row<T, VEC>& row) {
    using C = typename Cx<T>::type;
    bool ok = true;
    if (j < 0) { if (g.bc_y) ok = false; else j += g.ny; }
    else if (j >= g.ny) { if (g.bc_y) ok = false; else j -= g.ny; }
    const C* p = plane + (size_t)j * g.nx;
    const C zero = mk<T>(T(0), T(0));
    if (ok && c.active) ld_c<VEC>(p + c.x0, row.c);
    else {
#pragma unroll
        for (int i = 0; i < VEC; ++i) row.c[i] = zero;
    }
    row.el = (ok && c.l_load) ? p[c.xl] : zero;
    row.er = (ok && c.r_load) ? p[c.xr] : zero;
}

template <typename T, int VEC>
__device__ __forceinline__ typename Cx<T>::type west_of(const Row<T, VEC>& r, const Cols& c) {
    const auto s = shfl_up1(r.c[VEC - 1]);
    return c.l_shfl ? s : r.el;
}
template <typename T, int VEC>
__device__ __forceinline__ typename Cx<T>::type east_of(const Row<T, VEC>& r, const Cols& c) {
    const auto s = shfl_dn1(r.c[0]);
    return c.r_shfl ? s : r.er;
}

// Row-local (non-stencil) inputs of one component, prefetched one row ahead.
template <typename T, int VEC, bool RES>
struct Aux {
    typename Cx<T>::type psi[VEC];   // state psi (stages 2, 3)
    typename Cx<T>::type acc[VEC];   // running sum (stages 3, 4)
    T nin[VEC];                      // reservoir stage input (stage 1: the state n)
    T n[VEC];                        // reservoir state (stages 2, 3; stage 4 with noise: n_t)
    T nacc[VEC];                     // reservoir running sum (stages 3, 4)
};

template <typename T, int VEC>
struct AuxShared {
    T V[VEC];
    T P[VEC];
    typename Cx<T>::type E[VEC];
};

// Resident CTAs the register budget is sized for where the default allocation leaves bandwidth on the table
// (measured: spinor fp32 71 % -> 74 % of the HBM copy bandwidth with 4, scalar fp64 74 % -> 79 % with 6).
#ifndef PHX_STAGE_MINB_SPINOR
#define PHX_STAGE_MINB_SPINOR 4
#endif
#ifndef PHX_STAGE_MINB_F32
#define PHX_STAGE_MINB_F32 1
#endif
#ifndef PHX_STAGE_MINB_F64
#define PHX_STAGE_MINB_F64 6
#endif
template <typename T, int VEC, int MODEL, int STAGE, bool NOISE>
__global__ void __launch_bounds__(128, (model_spinor(MODEL) && sizeof(T) == 4) ? PHX_STAGE_MINB_SPINOR
                                       : (MODEL == M_SCALAR ? (sizeof(T) == 8 ? PHX_STAGE_MINB_F64 : PHX_STAGE_MINB_F32) : 1))
stage_kernel(const __grid_constant__ StageArgs<T> a) {
    using C = typename Cx<T>::type;
    constexpr bool SPINOR = model_spinor(MODEL);
    constexpr bool RES = model_reservoir(MODEL);
    constexpr int NC = SPINOR ? 2 : 1;
    const Geom& g = a.geo;
    const Coef<T>& k = a.k;

    const Cols col = make_cols<VEC>(g);
    const int j0 = (blockIdx.y * blockDim.y + threadIdx.y) * g.rows;
    const int j1 = min(j0 + g.rows, g.ny);
    const size_t boff = (size_t)blockIdx.z * g.plane;

    // ---- step counter bookkeeping ("step counter") ----------------------
    const uint64_t step = STAGE == 4 ? a.f.step[1] - 1 : a.f.step[0];
    if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0 && threadIdx.y == 0) {
        if (STAGE == 1) a.f.step[1] = step + 1;
        if (STAGE == 4) a.f.step[0] = step + 1;
    }
    if (j0 >= g.ny) return;   // whole warp row-chunk out of range (uniform per warp: threadIdx.y is per-warp-row)

    // ---- stage wiring -------------------------------------------------------------------------
    const C* yin[NC]; C* yout[NC]; const C* psi[NC]; C* acc[NC];
    const T* nin[NC]; T* nout[NC]; T* nst[NC]; T* nacc[NC];
#pragma unroll
    for (int s = 0; s < NC; ++s) {
        psi[s] = a.f.psi[s] + boff;
        acc[s] = a.f.acc[s] + boff;
        yin[s] = (STAGE == 1 ? a.f.psi[s] : (STAGE == 3 ? a.f.yb[s] : a.f.ya[s])) + boff;     // y2, y4 in ya; y3 in yb
        yout[s] = (STAGE == 4 ? a.f.psi[s] : (STAGE == 2 ? a.f.yb[s] : a.f.ya[s])) + boff;
        if constexpr (RES) {
            nst[s] = a.f.n[s] + boff;
            nacc[s] = a.f.nacc[s] + boff;
            nin[s] = (STAGE == 1 ? a.f.n[s] : (STAGE == 3 ? a.f.nb[s] : a.f.na[s])) + boff;
            nout[s] = (STAGE == 4 ? a.f.n[s] : (STAGE == 2 ? a.f.nb[s] : a.f.na[s])) + boff;
        }
    }
    const T a_dt = STAGE == 3 ? k.dt : k.hdt;          // a_s dt of Eqs. (3)-(5)
    const T w_dt = (STAGE == 1 || STAGE == 4) ? k.dt6 : k.dt3;   // weight of K_s in Eq. (6)

    // drive phase exp(-i omega t_s), t_s = (step + c_s) dt, evaluated in double
    T ph_re = T(1), ph_im = T(0);
    if (a.f.E != nullptr) {
        const double cs = STAGE == 1 ? 0.0 : (STAGE == 4 ? 1.0 : 0.5);
        const double t = ((double)step + cs) * k.dt_d;
        double sn, cn;
        sincos(-k.omega * t, &sn, &cn);
        ph_re = (T)cn; ph_im = (T)sn;
    }

    auto load_aux = [&](int j, Aux<T, VEC, RES> (&ax)[NC], AuxShared<T, VEC>& sh) {
        const size_t o = (size_t)j * g.nx + col.x0;
#pragma unroll
        for (int i = 0; i < VEC; ++i) { sh.V[i] = T(0); sh.P[i] = T(0); sh.E[i] = mk<T>(T(0), T(0)); }
        if (!col.active) return;
        if (a.f.V) ld_r<VEC>(a.f.V + o, sh.V);
        if (RES && a.f.P) ld_r<VEC>(a.f.P + o, sh.P);
        if (a.f.E) ld_c<VEC>(a.f.E + o, sh.E);
#pragma unroll
        for (int s = 0; s < NC; ++s) {
            if (STAGE == 2 || STAGE == 3) ld_c<VEC>(psi[s] + o, ax[s].psi);
            if (STAGE == 3 || STAGE == 4) ld_c<VEC>(acc[s] + o, ax[s].acc);
            if constexpr (RES) {
                ld_r<VEC>(nin[s] + o, ax[s].nin);
                if (STAGE == 2 || STAGE == 3 || (STAGE == 4 && NOISE)) ld_r<VEC>(nst[s] + o, ax[s].n);
                if (STAGE == 3 || STAGE == 4) ld_r<VEC>(nacc[s] + o, ax[s].nacc);
            }
        }
    };

    // DRAM -> L2 prefetch of everything row j of this thread's columns will read (no registers are tied up; the loads one
    // row ahead then hit L2).  The per-stage kernels are bound by HBM latency x bytes in flight: stage 1 moves 20 B per cell
    // and a thread has 24 B in flight with the register prefetch alone.
    constexpr int PFR = SPINOR ? (STAGE == 1 ? PHX_STAGE_PF_ROWS_SPINOR1 : PHX_STAGE_PF_ROWS_SPINOR) : PHX_STAGE_PF_ROWS;
    auto prefetch_row = [&](int j) {
        if (PFR <= 0 || !g.pf || !col.active || j >= j1) return;
        const size_t o = (size_t)j * g.nx + col.x0;
        auto pf = [](const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); };
#pragma unroll
        for (int s = 0; s < NC; ++s) {
            pf(yin[s] + o);
            if (STAGE == 2 || STAGE == 3) pf(psi[s] + o);
            if (STAGE == 3 || STAGE == 4) pf(acc[s] + o);
            if constexpr (RES) {
                pf(nin[s] + o);
                if (STAGE == 2 || STAGE == 3 || (STAGE == 4 && NOISE)) pf(nst[s] + o);
                if (STAGE == 3 || STAGE == 4) pf(nacc[s] + o);
            }
        }
        if (a.f.V) pf(a.f.V + o);
        if (RES && a.f.P) pf(a.f.P + o);
        if (a.f.E) pf(a.f.E + o);
    };
#pragma unroll 1
    for (int d = 2; d < 2 + PFR; ++d) prefetch_row(j0 + d);

    // ---- prologue: rows j0-1, j0, j0+1 of the stage input; row-local inputs of row j0 ---------
    Row<T, VEC> win[NC][4];
#pragma unroll
    for (int s = 0; s < NC; ++s) {
        load_row<T, VEC>(yin[s], j0 - 1, g, col, win[s][0]);
        load_row<T, VEC>(yin[s], j0, g, col, win[s][1]);
        load_row<T, VEC>(yin[s], j0 + 1, g, col, win[s][2]);
    }
    Aux<T, VEC, RES> cur[NC], nxt[NC];
    AuxShared<T, VEC> shc, shn;
    load_aux(j0, cur, shc);

    for (int j = j0; j < j1; ++j) {
        prefetch_row(j + 2 + PFR);
        // prefetch: stencil row j+2 and the row-local inputs of row j+1
        if (j + 1 < j1) {
#pragma unroll
            for (int s = 0; s < NC; ++s) load_row<T, VEC>(yin[s], j + 2, g, col, win[s][3]);
            load_aux(j + 1, nxt, shn);
        }

        // x neighbours of the rows in the window
        C cw[NC][3], ce[NC][3];   // west / east of rows j-1, j, j+1 (rows 0 and 2 only needed by TE-TM)
#pragma unroll
        for (int s = 0; s < NC; ++s) {
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                if (SPINOR || r == 1) {
                    cw[s][r] = west_of<T, VEC>(win[s][r], col);
                    ce[s][r] = east_of<T, VEC>(win[s][r], col);
                }
            }
        }

        C yn[NC][VEC], accn[NC][VEC];
        T nn[NC][VEC], naccn[NC][VEC];
#pragma unroll
        for (int s = 0; s < NC; ++s) {
            const int o_ = SPINOR ? 1 - s : 0;
#pragma unroll
            for (int i = 0; i < VEC; ++i) {
                const C y = win[s][1].c[i];
                const C yW = (i == 0) ? cw[s][1] : win[s][1].c[i - 1];
                const C yE = (i == VEC - 1) ? ce[s][1] : win[s][1].c[i + 1];
                const C yS = win[s][0].c[i];
                const C yN = win[s][2].c[i];
                const T rho = y.x * y.x + y.y * y.y - k.doff;
                const T nres = RES ? cur[s].nin[i] : T(0);

                // (hbar/2m) lap, Eq. (8)
                const T Lr = k.cx * (yE.x + yW.x - T(2) * y.x) + k.cy * (yN.x + yS.x - T(2) * y.x);
                const T Li = k.cx * (yE.y + yW.y - T(2) * y.y) + k.cy * (yN.y + yS.y - T(2) * y.y);

                T pot = shc.V[i] + k.g * rho;
                if (RES) pot += k.gr * nres;
                if (SPINOR) {
                    const C oc = win[o_][1].c[i];
                    pot += k.gx * (oc.x * oc.x + oc.y * oc.y - k.doff);
                }
                const T W = k.ih * pot;
                const T gain = RES ? (T(0.5) * k.Rr * nres - k.hgc) : -k.hgc;

                // K = i L - i W y + gain y
                T Kr = -Li + W * y.y + gain * y.x;
                T Ki = Lr - W * y.x + gain * y.y;

                if (SPINOR) {
                    // -(i/hbar) Delta_LT (d_xx - d_yy -+ 2 i d_xy) psi_other, compact nine-point form
                    const C oc = win[o_][1].c[i];
                    const C oW = (i == 0) ? cw[o_][1] : win[o_][1].c[i - 1];
                    const C oE = (i == VEC - 1) ? ce[o_][1] : win[o_][1].c[i + 1];
                    const C oS = win[o_][0].c[i], oN = win[o_][2].c[i];
                    const C oSW = (i == 0) ? cw[o_][0] : win[o_][0].c[i - 1];
                    const C oSE = (i == VEC - 1) ? ce[o_][0] : win[o_][0].c[i + 1];
                    const C oNW = (i == 0) ? cw[o_][2] : win[o_][2].c[i - 1];
                    const C oNE = (i == VEC - 1) ? ce[o_][2] : win[o_][2].c[i + 1];
                    const T dxx_r = oE.x + oW.x - T(2) * oc.x, dxx_i = oE.y + oW.y - T(2) * oc.y;
                    const T dyy_r = oN.x + oS.x - T(2) * oc.x, dyy_i = oN.y + oS.y - T(2) * oc.y;
                    const T dxy_r = oNE.x - oSE.x - oNW.x + oSW.x, dxy_i = oNE.y - oSE.y - oNW.y + oSW.y;
                    const T sgn = s == 0 ? T(-1) : T(1);
                    const T Jr = k.bxx * dxx_r - k.byy * dyy_r - sgn * k.bxy * dxy_i;
                    const T Ji = k.bxx * dxx_i - k.byy * dyy_i + sgn * k.bxy * dxy_r;
                    Kr += Ji;
                    Ki -= Jr;
                }
                if (a.f.E != nullptr) {
                    const T er = shc.E[i].x * ph_re - shc.E[i].y * ph_im;
                    const T ei = shc.E[i].x * ph_im + shc.E[i].y * ph_re;
                    Kr += k.ih * ei;
                    Ki -= k.ih * er;
                }
                T Kn = T(0);
                if (RES) Kn = shc.P[i] - (k.gamr + k.Rr * rho) * nres;

                // ---- fused Runge-Kutta sums, Eqs. (3)-(6) ---------------------------------------
                const C p = STAGE == 1 ? y : cur[s].psi[i];     // psi(t)
                if (STAGE == 1) {
                    yn[s][i] = mk<T>(p.x + a_dt * Kr, p.y + a_dt * Ki);
                    if (RES) nn[s][i] = nres + a_dt * Kn;
                } else if (STAGE == 2) {
                    yn[s][i] = mk<T>(p.x + a_dt * Kr, p.y + a_dt * Ki);
                    // acc = psi + dt6 K1 + dt3 K2 with dt6 K1 = r13 (y2 - psi): K1 is not re-read
                    // r13 + r13lo carries dt6 / hdt to twice the precision of T, so the weight of K1 is the canonical dt6.  The two
                    // increments are summed FIRST and added to psi in one rounding: psi + (y2 - psi)/3 on its own lands on a
                    // lattice of thirds of an ulp of psi (psi and y2 are both floats), and rounding that lattice to T is biased
                    // along K1 by 0.03 ulp per step -- a phase error that grew linearly (1.5e-5 after 10^4 fp32 steps, measured).
                    const T dx_ = y.x - p.x, dy_ = y.y - p.y;
                    accn[s][i] = mk<T>(p.x + fma(k.r13, dx_, fma(k.r13lo, dx_, w_dt * Kr)), p.y + fma(k.r13, dy_, fma(k.r13lo, dy_, w_dt * Ki)));
                    if (RES) {
                        const T n0 = cur[s].n[i];
                        nn[s][i] = n0 + a_dt * Kn;
                        const T dn_ = nres - n0;
                        naccn[s][i] = n0 + fma(k.r13, dn_, fma(k.r13lo, dn_, w_dt * Kn));
                    }
                } else if (STAGE == 3) {
                    yn[s][i] = mk<T>(p.x + a_dt * Kr, p.y + a_dt * Ki);
                    accn[s][i] = mk<T>(cur[s].acc[i].x + w_dt * Kr, cur[s].acc[i].y + w_dt * Ki);
                    if (RES) {
                        nn[s][i] = cur[s].n[i] + a_dt * Kn;
                        naccn[s][i] = cur[s].nacc[i] + w_dt * Kn;
                    }
                } else {
                    C out = mk<T>(cur[s].acc[i].x + w_dt * Kr, cur[s].acc[i].y + w_dt * Ki);
                    if (RES) nn[s][i] = cur[s].nacc[i] + w_dt * Kn;
                    if (NOISE) {
                        // dW of Eq. (22): variance sig2 (gamma_c + R n_t) per real component
                        const uint32_t cell = (uint32_t)j * (uint32_t)g.nx + (uint32_t)(col.x0 + i);   // < 2^32 (desc_ok), unsigned product
                        const uint4 w = noise_words(a.seed, blockIdx.z, step, cell);
                        const C xi = s == 0 ? normal_pair(w.x, w.y, T(0)) : normal_pair(w.z, w.w, T(0));
                        const T nt = RES ? cur[s].n[i] : T(0);
                        const T sigma = sqrt(k.sig2 * (T(2) * k.hgc + k.Rr * nt));
                        out.x += sigma * xi.x;
                        out.y += sigma * xi.y;
                    }
                    yn[s][i] = out;
                }
            }
        }

        // ---- stores ---------------------------------------------------------------------------
        if (col.active) {
            const size_t o = (size_t)j * g.nx + col.x0;
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                st_c<VEC>(yout[s] + o, yn[s]);
                if (STAGE == 2 || STAGE == 3) st_c<VEC>(acc[s] + o, accn[s]);
                if constexpr (RES) {
                    st_r<VEC>(nout[s] + o, nn[s]);
                    if (STAGE == 2 || STAGE == 3) st_r<VEC>(nacc[s] + o, naccn[s]);
                }
            }
        }

        // ---- slide the window -------------------------------------------------------------------
#pragma unroll
        for (int s = 0; s < NC; ++s) {
            win[s][0] = win[s][1];
            win[s][1] = win[s][2];
            win[s][2] = win[s][3];
            cur[s] = nxt[s];
        }
        shc = shn;
    }
}

}  // namespace phx
