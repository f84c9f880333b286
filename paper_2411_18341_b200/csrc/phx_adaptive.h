// phx_adaptive.h -- device control block, kernel arguments and host entry points of the adaptive Dormand-Prince 5(4)
// integrator (phx_adaptive.cu; reading Q20).  Internal to libphx.
#pragma once

#include "phx_common.cuh"

namespace phx {

// Capacity of the on-device attempt log (one record per attempt of the last phx_step_adaptive call).
constexpr int DP_LOG_CAP = 1 << 16;

// Lives in the workspace; written by the one-thread setup / control kernels, read by every stage kernel.
struct DpCtl {
    // call parameters (copied in by the host before the graph launch)
    double t_end, atol, rtol, h_init, h_min, h_max;
    long long max_attempts;
    // integrator state (persists from call to call)
    double t;                       // current time
    double h;                       // step size the next attempt proposes (<= 0: use h_init)
    long long n_accept, n_reject;
    int cur;                        // which state buffer holds u: 0 = psi / n, 1 = acc / nacc
    int k1_valid;                   // K_1 holds f(u, t) (the K_7 of the last accepted step: FSAL)
    // the attempt in flight
    double hu;                      // step actually tried (clipped at t_end, rounded once to T)
    int clipped, done;
    unsigned long long err_bits;    // bit pattern of the error norm (atomicMax target)
    double err_last;
    long long attempts;             // attempts of this call
    long long log_count;
    int* log_accept;
    int* log_q;
    double* log_h;
    double* log_err;
};

template <typename T>
struct DpArgs {
    using C = typename Cx<T>::type;
    Geom geo;
    Coef<T> k;
    C* S[2][2];          // state buffers [cur][component]: 0 = psi, 1 = acc
    C* Y[2][2];          // stage-input ping-pong [which][component]: ya, yb
    C* K[7][2];          // K_1..K_7 [stage][component]
    T* Sn[2][2];         // reservoir: n, nacc
    T* Yn[2][2];         // na, nb
    T* Kn[7][2];
    const T* V;
    const T* P;
    const C* E;
    DpCtl* ctl;
    T c[7], a[7][7], e[7];   // Dormand-Prince tableau, each coefficient rounded once to T
};

template <typename T> cudaError_t dp_launch_attempt(const DpArgs<T>& a, int model, cudaStream_t st);
template <typename T> cudaError_t dp_launch_finalize(const DpArgs<T>& a, int model, int n_sm, cudaStream_t st);
cudaError_t dp_launch_setup(DpCtl* c, unsigned long long handle, int prec32, cudaStream_t st);
cudaError_t dp_launch_control(DpCtl* c, unsigned long long handle, int prec32, int log_cap, cudaStream_t st);

}  // namespace phx
