// phx_step.cuh -- variant STEP: one kernel per RK4 step, the four stages temporally blocked on chip
// (DESIGN.md section 5.2).  The idea is the paper's subgrid decomposition with N_halo = 4 (PAPER.md:167-173,
// :183: a whole time step on a haloed subgrid is independent of its neighbours), re-designed for B200:
// the "subgrid" is a warp-wide column strip that streams down y, and the haloed data live in REGISTERS.
//
// One warp owns a strip of W = 32*VEC columns (VEC cells per lane, one 128-bit load for complex fp32 pairs)
// of which the inner W-8 are output columns, and walks a chunk of rows.  The four stages run as a software
// pipeline along y: in the iteration whose front row is j,
//     stage 1 evaluates K1 on row j   from psi rows j-1..j+1  -> y2[j]   = psi + dt/2 K1, acc  = psi + dt/6 K1
//     stage 2 evaluates K2 on row j-1 from y2  rows j-2..j    -> y3[j-1] = psi + dt/2 K2, acc += dt/3 K2
//     stage 3 evaluates K3 on row j-2 from y3  rows j-3..j-1  -> y4[j-2] = psi + dt   K3, acc += dt/3 K3
//     stage 4 evaluates K4 on row j-3 from y4  rows j-4..j-2  -> psi(t+dt)[j-3] = acc + dt/6 K4 (+ dW, Eq. (22))
// (Eqs. (2)-(6)).  Every stage input is a three-row register window per lane; x neighbours
// come from warp shuffles, so there is no shared memory and no block-level barrier.  The four halo columns
// on each side of the strip are recomputed redundantly (their lanes compute values that are never stored;
// each stage invalidates one more column from either edge), the 4+4 halo rows of a chunk likewise.
// HBM traffic per cell-step: read psi, V once, write psi once (+ halo re-reads, mostly L2 hits) instead of the
// 14 complex transfers of variant STAGE.  psi(t) and psi(t+dt) are distinct buffers (ping-pong).
#pragma once

#include "phx_common.cuh"
#include "phx_deriv.cuh"
#include "phx_philox.cuh"

#ifndef PHX_STEP_UNROLL
#define PHX_STEP_UNROLL 4
#endif
#ifndef PHX_STEP_PF_ROWS
#define PHX_STEP_PF_ROWS 6
#endif

namespace phx {

template <typename T>
struct StepArgs {
    using C = typename Cx<T>::type;
    Geom geo;
    Coef<T> k;
    const C* psi_in[2];
    C* psi_out[2];
    const T* n_in[2];
    T* n_out[2];
    const T* V;                 // [ny][nx] or nullptr
    const T* P;                 // [ny][nx] or nullptr
    const uint64_t* step_in;    // completed steps before this one
    uint64_t* step_out;         // receives step_in + 1 (the slot the next launch reads)
    uint32_t seed;
    int ly;                     // rows per chunk
    int strips;                 // strips per row of the grid
};

namespace stepk {

template <int VEC> __device__ __forceinline__ void ldc(const float2* p, float2 (&v)[VEC]) {
    if constexpr (VEC == 2) { const float4 q = __ldg(reinterpret_cast<const float4*>(p)); v[0] = make_float2(q.x, q.y); v[1] = make_float2(q.z, q.w); }
    else v[0] = __ldg(p);
}
template <int VEC> __device__ __forceinline__ void ldc(const double2* p, double2 (&v)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) v[i] = __ldg(p + i);
}
template <int VEC> __device__ __forceinline__ void stc(float2* p, const float2 (&v)[VEC]) {
    if constexpr (VEC == 2) *reinterpret_cast<float4*>(p) = make_float4(v[0].x, v[0].y, v[1].x, v[1].y);
    else *p = v[0];
}
template <int VEC> __device__ __forceinline__ void stc(double2* p, const double2 (&v)[VEC]) {
#pragma unroll
    for (int i = 0; i < VEC; ++i) p[i] = v[i];
}
template <int VEC> __device__ __forceinline__ void ldr(const float* p, float (&v)[VEC]) {
    if constexpr (VEC == 2) { const float2 q = __ldg(reinterpret_cast<const float2*>(p)); v[0] = q.x; v[1] = q.y; }
    else v[0] = __ldg(p);
}
template <int VEC> __device__ __forceinline__ void ldr(const double* p, double (&v)[VEC]) {
    if constexpr (VEC == 2) { const double2 q = __ldg(reinterpret_cast<const double2*>(p)); v[0] = q.x; v[1] = q.y; }
    else v[0] = __ldg(p);
}
template <int VEC> __device__ __forceinline__ void str(float* p, const float (&v)[VEC]) {
    if constexpr (VEC == 2) *reinterpret_cast<float2*>(p) = make_float2(v[0], v[1]);
    else *p = v[0];
}
template <int VEC> __device__ __forceinline__ void str(double* p, const double (&v)[VEC]) {
    if constexpr (VEC == 2) *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
    else *p = v[0];
}

// DRAM -> L2 prefetch of the line holding p (no register is tied up; the register fetch one row ahead then hits L2).
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

__device__ __forceinline__ float2 up1(float2 v) { return make_float2(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ float2 dn1(float2 v) { return make_float2(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ double2 up1(double2 v) { return make_double2(__shfl_up_sync(0xffffffffu, v.x, 1), __shfl_up_sync(0xffffffffu, v.y, 1)); }
__device__ __forceinline__ double2 dn1(double2 v) { return make_double2(__shfl_down_sync(0xffffffffu, v.x, 1), __shfl_down_sync(0xffffffffu, v.y, 1)); }

// Three-row window of one component's stage input: r[0] = row below the centre (j-1), r[1] = centre, r[2] = j+1.
template <typename T, int VEC>
struct Win3 {
    typename Cx<T>::type r[3][VEC];
};

// Neighbourhood of cell i of the centre row of a window; west/east of the lane's cells by shuffle.
// NINE = false leaves the corners unset (scalar models never read them).
template <typename T, int VEC, bool NINE>
__device__ __forceinline__ void gather(const Win3<T, VEC>& w, Nbhd<T> (&nb)[VEC]) {
    using C = typename Cx<T>::type;
    C west[3], east[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        if (NINE || r == 1) {
            west[r] = up1(w.r[r][VEC - 1]);
            east[r] = dn1(w.r[r][0]);
        }
    }
#pragma unroll
    for (int i = 0; i < VEC; ++i) {
        nb[i].c = w.r[1][i];
        nb[i].s = w.r[0][i];
        nb[i].n = w.r[2][i];
        nb[i].w = i == 0 ? west[1] : w.r[1][i - 1];
        nb[i].e = i == VEC - 1 ? east[1] : w.r[1][i + 1];
        if (NINE) {
            nb[i].sw = i == 0 ? west[0] : w.r[0][i - 1];
            nb[i].se = i == VEC - 1 ? east[0] : w.r[0][i + 1];
            nb[i].nw = i == 0 ? west[2] : w.r[2][i - 1];
            nb[i].ne = i == VEC - 1 ? east[2] : w.r[2][i + 1];
        }
    }
}

}  // namespace stepk

template <typename T, int VEC, int MODEL, bool NOISE, bool ZBC, int MINB>
__global__ void __launch_bounds__(128, MINB)
step_kernel(const __grid_constant__ StepArgs<T> a) {
    using namespace stepk;
    using C = typename Cx<T>::type;
    constexpr bool SPINOR = model_spinor(MODEL);
    constexpr bool RES = model_reservoir(MODEL);
    constexpr int NC = SPINOR ? 2 : 1;
    constexpr int W = 32 * VEC, OUTW = W - 8;
    const Geom& g = a.geo;
    const Coef<T>& k = a.k;
    const int nx = g.nx, ny = g.ny;

    const int lane = threadIdx.x & 31;
    const int strip = blockIdx.x * 4 + (threadIdx.x >> 5);
    const uint64_t step = *a.step_in;
    if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0) *a.step_out = step + 1;
    if (strip >= a.strips) return;   // warp-uniform

    // ---- columns of this lane ----------------------------------------------------------------------------------
    const int xl = strip * OUTW - 4 + lane * VEC;   // unwrapped column of the lane's first cell
    int xg = xl;                                     // column actually addressed
    bool inx = true;                                 // false: outside a zero boundary
    if (xl < 0 || xl >= nx) {
        if (ZBC && g.bc_x) { inx = false; xg = 0; }
        else { xg = xl % nx; if (xg < 0) xg += nx; }
    }
    const bool st_lane = lane * VEC >= 4 && lane * VEC < W - 4 && xl < nx;   // lane owns output columns

    // ---- rows of this chunk ------------------------------------------------------------------------------------
    const int r0 = blockIdx.y * a.ly;
    const int r1 = min(r0 + a.ly, ny);
    const size_t boff = (size_t)blockIdx.z * g.plane;
    const bool zy = ZBC && g.bc_y;

    // ---- register windows (state carried from one iteration to the next; row numbers relative to the front j) ----
    const C czero = mk<T>(T(0), T(0));
    C psw[NC][4][VEC];                      // psi rows j-2, j-1, j, j+1
    C psn[NC][VEC];                         // psi row j+2, in flight
    Win3<T, VEC> y2[NC], y3[NC], y4[NC];    // r[0], r[1]: rows (j-2, j-1), (j-3, j-2), (j-4, j-3); r[2] is produced in the iteration
    C acc[NC][3][VEC];                      // running sum of Eq. (6), rows j-1, j-2, j-3
    T Vw[4][VEC], Pw[4][VEC];               // V, P rows j, j-1, j-2, j-3
    T Vn[VEC], Pn[VEC];                     // row j+1, in flight
    T nw[NC][4][VEC], nn[NC][VEC];          // reservoir state rows j, j-1, j-2, j-3; row j+1 in flight
    T n2[NC][VEC], n3[NC][VEC], n4[NC][VEC];   // reservoir stage inputs of rows j-1, j-2, j-3 (cell-local)
    T nacc[NC][3][VEC];                     // reservoir running sum, rows j-1, j-2, j-3
#pragma unroll
    for (int s = 0; s < NC; ++s) {
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
#pragma unroll
            for (int r = 0; r < 4; ++r) { psw[s][r][i] = czero; nw[s][r][i] = T(0); }
#pragma unroll
            for (int r = 0; r < 3; ++r) { y2[s].r[r][i] = czero; y3[s].r[r][i] = czero; y4[s].r[r][i] = czero; acc[s][r][i] = czero; nacc[s][r][i] = T(0); }
            psn[s][i] = czero; nn[s][i] = T(0); n2[s][i] = T(0); n3[s][i] = T(0); n4[s][i] = T(0);
        }
    }
#pragma unroll
    for (int i = 0; i < VEC; ++i) {
#pragma unroll
        for (int r = 0; r < 4; ++r) { Vw[r][i] = T(0); Pw[r][i] = T(0); }
        Vn[i] = T(0); Pn[i] = T(0);
    }

    // wrapped index of the psi row fetched in the first iteration (row r0-4); advanced by one per iteration
    int qw = r0 - 4;
    if (!zy) { qw %= ny; if (qw < 0) qw += ny; }
    int qprev = 0;          // wrapped index of the row fetched in the previous iteration (= row j+1 now)
    bool okprev = false;
    // rows further ahead are pulled from DRAM into L2 by prefetch instructions (PF_ROWS ahead of the register fetch)
    constexpr int PF_ROWS = PHX_STEP_PF_ROWS;
    constexpr int UNROLL_J = PHX_STEP_UNROLL;
    int qpf = r0 - 4 + PF_ROWS;
    if (!zy) { qpf %= ny; if (qpf < 0) qpf += ny; }
    if (PF_ROWS > 0 && inx) {
        // warm-up: the first PF_ROWS rows of the chunk
        int q = r0 - 4;
        if (!zy) { q %= ny; if (q < 0) q += ny; }
        for (int r = 0; r < PF_ROWS; ++r) {
            if (!zy || (q >= 0 && q < ny)) {
                const size_t o = (size_t)q * nx + xg;
#pragma unroll
                for (int s = 0; s < NC; ++s) {
                    prefetch_l2(a.psi_in[s] + boff + o);
                    if (RES) prefetch_l2(a.n_in[s] + boff + o);
                }
                if (a.V) prefetch_l2(a.V + o);
                if (RES && a.P) prefetch_l2(a.P + o);
            }
            ++q;
            if (!zy && q == ny) q = 0;
        }
    }

#pragma unroll UNROLL_J
    for (int j = r0 - 6; j <= r1 + 2; ++j) {
        if (PF_ROWS > 0) {
            if (inx && (j + 2 + PF_ROWS <= r1 + 3) && (!zy || (qpf >= 0 && qpf < ny))) {
                const size_t o = (size_t)qpf * nx + xg;
#pragma unroll
                for (int s = 0; s < NC; ++s) {
                    prefetch_l2(a.psi_in[s] + boff + o);
                    if (RES) prefetch_l2(a.n_in[s] + boff + o);
                }
                if (a.V) prefetch_l2(a.V + o);
                if (RES && a.P) prefetch_l2(a.P + o);
            }
            ++qpf;
            if (!zy && qpf == ny) qpf = 0;
        }
        // ---- fetch: psi row j+2; row-local inputs (V, P, n) of row j+1 -----------------------------------------------
        const bool okq = inx && (j + 2 <= r1 + 3) && (!zy || (qw >= 0 && qw < ny));
        {
            const size_t o = (size_t)qw * nx + xg;
#pragma unroll
            for (int s = 0; s < NC; ++s) {
#pragma unroll
                for (int i = 0; i < VEC; ++i) psn[s][i] = czero;
                if (okq) ldc<VEC>(a.psi_in[s] + boff + o, psn[s]);
            }
            const size_t op = (size_t)qprev * nx + xg;
#pragma unroll
            for (int i = 0; i < VEC; ++i) { Vn[i] = T(0); Pn[i] = T(0); }
            if (okprev) {
                if (a.V) ldr<VEC>(a.V + op, Vn);
                if (RES && a.P) ldr<VEC>(a.P + op, Pn);
            }
            if constexpr (RES) {
#pragma unroll
                for (int s = 0; s < NC; ++s) {
#pragma unroll
                    for (int i = 0; i < VEC; ++i) nn[s][i] = T(0);
                    if (okprev) ldr<VEC>(a.n_in[s] + boff + op, nn[s]);
                }
            }
        }

        C accN[NC][VEC];
        T n2N[NC][VEC], n3N[NC][VEC], n4N[NC][VEC], naccN[NC][VEC];
#pragma unroll
        for (int s = 0; s < NC; ++s) {
#pragma unroll
            for (int i = 0; i < VEC; ++i) { accN[s][i] = czero; n2N[s][i] = T(0); n3N[s][i] = T(0); n4N[s][i] = T(0); naccN[s][i] = T(0); }
        }

        if (j >= r0 - 3) {
            // in-domain flags of the rows whose next stage input is written (zero boundaries: 0 outside the grid)
            const bool in1 = !ZBC || (inx && (!zy || (j >= 0 && j < ny)));
            const bool in2 = !ZBC || (inx && (!zy || (j - 1 >= 0 && j - 1 < ny)));
            const bool in3 = !ZBC || (inx && (!zy || (j - 2 >= 0 && j - 2 < ny)));
            Nbhd<T> nb[NC][VEC];
            Diff<T> df[NC][VEC];
            auto O = [](int s) { return SPINOR ? 1 - s : 0; };            // index of the other component
            auto diffs = [](const Nbhd<T> (&nb)[NC][VEC], Diff<T> (&df)[NC][VEC]) {
#pragma unroll
                for (int s = 0; s < NC; ++s) {
#pragma unroll
                    for (int i = 0; i < VEC; ++i) differences<T, SPINOR>(nb[s][i], df[s][i]);
                }
            };

            // ---- stage 1: K1 on row j from psi rows j-1, j, j+1 (Eq. (2)) ---------------------------------------------
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                Win3<T, VEC> w;
#pragma unroll
                for (int i = 0; i < VEC; ++i) { w.r[0][i] = psw[s][1][i]; w.r[1][i] = psw[s][2][i]; w.r[2][i] = psw[s][3][i]; }
                gather<T, VEC, SPINOR>(w, nb[s]);
            }
            diffs(nb, df);
#pragma unroll
            for (int s = 0; s < NC; ++s) {
#pragma unroll
                for (int i = 0; i < VEC; ++i) {
                    T Kn;
                    const T nres = RES ? nw[s][0][i] : T(0);
                    const C K = deriv<T, SPINOR, RES>(k, nb[s][i].c, df[s][i], nb[O(s)][i].c, df[O(s)][i], s == 0, nres, Vw[0][i], Pw[0][i], Kn);
                    const C p = psw[s][2][i];
                    y2[s].r[2][i] = in1 ? fma2s(k.hdt, K, p) : czero;
                    accN[s][i] = fma2s(k.dt6, K, p);
                    if (RES) { n2N[s][i] = nres + k.hdt * Kn; naccN[s][i] = nres + k.dt6 * Kn; }
                }
            }

            // ---- stage 2: K2 on row j-1 from y2 rows j-2, j-1, j (Eq. (3)) --------------------------------------------
#pragma unroll
            for (int s = 0; s < NC; ++s) gather<T, VEC, SPINOR>(y2[s], nb[s]);
            diffs(nb, df);
#pragma unroll
            for (int s = 0; s < NC; ++s) {
#pragma unroll
                for (int i = 0; i < VEC; ++i) {
                    T Kn;
                    const C K = deriv<T, SPINOR, RES>(k, nb[s][i].c, df[s][i], nb[O(s)][i].c, df[O(s)][i], s == 0, RES ? n2[s][i] : T(0), Vw[1][i], Pw[1][i], Kn);
                    const C p = psw[s][1][i];
                    y3[s].r[2][i] = in2 ? fma2s(k.hdt, K, p) : czero;
                    acc[s][0][i] = fma2s(k.dt3, K, acc[s][0][i]);
                    if (RES) { n3N[s][i] = nw[s][1][i] + k.hdt * Kn; nacc[s][0][i] += k.dt3 * Kn; }
                }
            }

            // ---- stage 3: K3 on row j-2 from y3 rows j-3, j-2, j-1 (Eq. (4)) ------------------------------------------
#pragma unroll
            for (int s = 0; s < NC; ++s) gather<T, VEC, SPINOR>(y3[s], nb[s]);
            diffs(nb, df);
#pragma unroll
            for (int s = 0; s < NC; ++s) {
#pragma unroll
                for (int i = 0; i < VEC; ++i) {
                    T Kn;
                    const C K = deriv<T, SPINOR, RES>(k, nb[s][i].c, df[s][i], nb[O(s)][i].c, df[O(s)][i], s == 0, RES ? n3[s][i] : T(0), Vw[2][i], Pw[2][i], Kn);
                    const C p = psw[s][0][i];
                    y4[s].r[2][i] = in3 ? fma2s(k.dt, K, p) : czero;
                    acc[s][1][i] = fma2s(k.dt3, K, acc[s][1][i]);
                    if (RES) { n4N[s][i] = nw[s][2][i] + k.dt * Kn; nacc[s][1][i] += k.dt3 * Kn; }
                }
            }

            // ---- stage 4: K4 on row j-3 from y4 rows j-4, j-3, j-2; psi(t+dt) of Eq. (6) (+ dW of Eq. (22)) ----------
#pragma unroll
            for (int s = 0; s < NC; ++s) gather<T, VEC, SPINOR>(y4[s], nb[s]);
            diffs(nb, df);
            const int jr = j - 3;
            const bool st_row = jr >= r0 && jr < r1;
#pragma unroll
            for (int s = 0; s < NC; ++s) {
                C out[VEC];
                T nout[VEC];
#pragma unroll
                for (int i = 0; i < VEC; ++i) {
                    T Kn;
                    const C K = deriv<T, SPINOR, RES>(k, nb[s][i].c, df[s][i], nb[O(s)][i].c, df[O(s)][i], s == 0, RES ? n4[s][i] : T(0), Vw[3][i], Pw[3][i], Kn);
                    out[i] = fma2s(k.dt6, K, acc[s][2][i]);
                    nout[i] = RES ? nacc[s][2][i] + k.dt6 * Kn : T(0);
                }
                if (st_row && st_lane) {
                    if (NOISE) {
#pragma unroll
                        for (int i = 0; i < VEC; ++i) {
                            const uint32_t cell = (uint32_t)jr * (uint32_t)nx + (uint32_t)(xl + i);
                            const uint4 wd = noise_words(a.seed, blockIdx.z, step, cell);
                            const C xi = s == 0 ? normal_pair(wd.x, wd.y, T(0)) : normal_pair(wd.z, wd.w, T(0));
                            const T nt = RES ? nw[s][3][i] : T(0);      // reservoir at the start of the step
                            const T sigma = sqrt(k.sig2 * (T(2) * k.hgc + k.Rr * nt));
                            out[i] = fma2s(sigma, xi, out[i]);
                        }
                    }
                    const size_t o = boff + (size_t)jr * nx + xl;
                    stc<VEC>(a.psi_out[s] + o, out);
                    if constexpr (RES) str<VEC>(a.n_out[s] + o, nout);
                }
            }
        }

        // ---- slide every window by one row -----------------------------------------------------------------------------
#pragma unroll
        for (int s = 0; s < NC; ++s) {
#pragma unroll
            for (int i = 0; i < VEC; ++i) {
                psw[s][0][i] = psw[s][1][i]; psw[s][1][i] = psw[s][2][i]; psw[s][2][i] = psw[s][3][i]; psw[s][3][i] = psn[s][i];
                y2[s].r[0][i] = y2[s].r[1][i]; y2[s].r[1][i] = y2[s].r[2][i];
                y3[s].r[0][i] = y3[s].r[1][i]; y3[s].r[1][i] = y3[s].r[2][i];
                y4[s].r[0][i] = y4[s].r[1][i]; y4[s].r[1][i] = y4[s].r[2][i];
                acc[s][2][i] = acc[s][1][i]; acc[s][1][i] = acc[s][0][i]; acc[s][0][i] = accN[s][i];
                if (RES) {
                    nw[s][3][i] = nw[s][2][i]; nw[s][2][i] = nw[s][1][i]; nw[s][1][i] = nw[s][0][i]; nw[s][0][i] = nn[s][i];
                    n4[s][i] = n4N[s][i]; n3[s][i] = n3N[s][i]; n2[s][i] = n2N[s][i];
                    nacc[s][2][i] = nacc[s][1][i]; nacc[s][1][i] = nacc[s][0][i]; nacc[s][0][i] = naccN[s][i];
                }
            }
        }
#pragma unroll
        for (int i = 0; i < VEC; ++i) {
            Vw[3][i] = Vw[2][i]; Vw[2][i] = Vw[1][i]; Vw[1][i] = Vw[0][i]; Vw[0][i] = Vn[i];
            Pw[3][i] = Pw[2][i]; Pw[2][i] = Pw[1][i]; Pw[1][i] = Pw[0][i]; Pw[0][i] = Pn[i];
        }
        qprev = qw;
        okprev = okq;
        ++qw;
        if (!zy && qw == ny) qw = 0;
    }
}

}  // namespace phx
