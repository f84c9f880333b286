// phx_common.cuh -- shared device-side types of libphx (sm_100a).  Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace phx {

// Interleaved complex of the working real type T (interleaved storage).
template <typename T> struct Cx;
template <> struct Cx<float> { using type = float2; };
template <> struct Cx<double> { using type = double2; };

template <typename T> __device__ __forceinline__ typename Cx<T>::type mk(T re, T im) {
    typename Cx<T>::type z; z.x = re; z.y = im; return z;
}

// Canonical coefficient set, each value rounded once to T on the host (DESIGN.md section 2,
// "step 0"); only exact factors (1/2, 2, 4) are pre-combined: hdt = dt/2.
template <typename T>
struct Coef {
    T cx, cy, ih, g, gx, gr, Rr, hgc, gamr, bxx, byy, bxy, dt, hdt, dt6, dt3, sig2, doff;
    T r13, r13lo;   // dt6 / hdt as an unevaluated sum of two T (hi + lo), used to rebuild dt6*K1 from y2 - psi (variant STAGE,
                    // DESIGN.md section 5.1): with one T the weight of K1 differs from the canonical dt6 by a relative 2^-25,
                    // a systematic error that grows linearly with the step count (3e-5 after 10^4 fp32 steps)
    double omega;   // drive frequency, phase evaluated in double
    double dt_d;    // dt as double (the T-rounded value widened), for t = step*dt
};

// Model switches (compile-time per kernel instantiation).
enum : int { M_SCALAR = 0, M_RESERVOIR = 1, M_SPINOR = 2, M_SPINOR_RESERVOIR = 3 };
__host__ __device__ constexpr bool model_spinor(int m) { return m == M_SPINOR || m == M_SPINOR_RESERVOIR; }
__host__ __device__ constexpr bool model_reservoir(int m) { return m == M_RESERVOIR || m == M_SPINOR_RESERVOIR; }

// All device pointers of one grid (planes of [batch][ny][nx]); index 0 = "+", 1 = "-".
template <typename T>
struct Fields {
    using C = typename Cx<T>::type;
    C* psi[2];      // state
    C* ya[2];       // stage ping
    C* yb[2];       // stage pong
    C* acc[2];      // running RK sum
    T* n[2];        // reservoir state
    T* na[2];
    T* nb[2];
    T* nacc[2];
    const T* V;     // [ny][nx] or nullptr
    const T* P;     // [ny][nx] or nullptr
    const C* E;     // [ny][nx] or nullptr
    uint64_t* step; // step[0] = completed steps (read by all stages), step[1] = scratch slot
};

struct Geom {
    int nx, ny, batch;
    int bc_x, bc_y;        // 0 periodic, 1 zero
    int rows;              // rows per CTA (variant STAGE)
    int pf;                // variant STAGE: 1 = prefetch rows ahead into L2 (working sets beyond L2 only)
    size_t plane;          // nx*ny
};

}  // namespace phx
