/*
 * phx_oracle.h -- C ABI of the CPU ORACLE for the PHOENIX RK4 hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference leg may load this library.  It shares no code with the CUDA
 * path under paper_2411_18341_b200/ and neither side includes or imports the other.
 *
 * The oracle follows /root/reference/PAPER.md step by step, in the paper's own unfused form
 * (separate K1..K4 buffers and a stage buffer, PAPER.md:100-144 Listing 1, :181 "six buffers"):
 *   - Eq. (1)  PAPER.md:25      damped nonlinear Schroedinger equation
 *   - Eqs. (2)-(6) PAPER.md:53-62  fixed-step RK4
 *   - Eq. (8)  PAPER.md:203     five-point Laplacian with separate dx, dy
 *   - Eqs. (16)-(17) PAPER.md:361-364  spinor, reservoir, TE-TM, coherent drive E, noise dW
 *   - Eq. (22) PAPER.md:454-456  complex Wiener noise covariance
 * All arithmetic is IEEE double, one thread, no FMA contraction, no blocking or fusion.
 * The readings taken where the paper is silent or garbled are listed in DESIGN.md section 3.
 *
 * Adaptive Dormand-Prince 5(4): orc_step_dp54 below (the paper names the method only).
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"): stencil vs. dense brute force and vs. its
 * Fourier symbol; plane-wave amplification R(z)^N; loss and norm closed forms; reduction of
 * plane-wave states to a 0-dimensional RK4 written independently in Python (nonlinearity,
 * reservoir, spinor, TE-TM, drive); reservoir-only closed form; sine eigenmodes for zero
 * boundaries; RK4 order test; Philox4x32-10 known-answer vectors; normal-map moments.
 * Parity unpinned: statistics of full noisy trajectories beyond the integer stream, the
 * normal map's moments and short segments (the dynamics are chaotic).
 */
#ifndef PHX_ORACLE_H
#define PHX_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Physical parameters, as in Eqs. (1), (16), (17), (22). */
typedef struct {
    double hbar, m;          /* Eq. (1) */
    double g;                /* same-spin nonlinearity g |psi_s|^2 */
    double g_x;              /* cross-spin nonlinearity g_x |psi_-s|^2, Eq. (16) */
    double g_r;              /* reservoir interaction g_r n, Eq. (16) */
    double R;                /* condensation rate, Eqs. (16), (17) */
    double gamma_c;          /* loss gamma of psi, Eq. (1) / (16) */
    double gamma_r;          /* reservoir loss, Eq. (17) */
    double beta;             /* Delta_LT of J = Delta_LT (d_x -+ i d_y)^2 */
    double dt;               /* RK4 step */
    double noise_scale;      /* nu, scales the Wiener noise variance */
    double density_offset;   /* 1/DeltaV of the renormalised density, PAPER.md:452 (0 = off) */
    double omega;            /* drive frequency: E(r,t) = E(r) exp(-i omega t) */
} orc_params;

/* Canonical derived coefficients ("step 0").  Each is evaluated in
 * double with exactly the expression in orc_derive_coeffs and then, when prec32 != 0,
 * rounded once to float and widened back. */
enum {
    ORC_CX = 0, ORC_CY, ORC_IH, ORC_G, ORC_GX, ORC_GR, ORC_RR, ORC_HGC, ORC_GAMR,
    ORC_BXX, ORC_BYY, ORC_BXY, ORC_DT, ORC_DT6, ORC_DT3, ORC_SIG2, ORC_DOFF, ORC_OMEGA,
    ORC_NCOEF
};

typedef struct {
    int32_t nx, ny, batch;       /* arrays are [batch][ny][nx], x fastest */
    int32_t spinor;              /* 0: psi_+ only; 1: psi_+ and psi_- */
    int32_t reservoir;           /* 0: n == 0;     1: n_+ (and n_- if spinor) integrated */
    int32_t noise;               /* 0/1: add dW after each step (Eq. 22) */
    int32_t bc_x, bc_y;          /* 0 periodic, 1 zero */
    uint32_t seed;               /* Philox key word 0 */
    double coef[ORC_NCOEF];
    const double* V;             /* [ny][nx] real, shared by the batch; NULL = 0 */
    const double* P;             /* [ny][nx] real pump P_+ = P_-; NULL = 0 */
    const double* E;             /* [ny][nx] complex drive amplitude E_+ = E_-; NULL = 0 */
    uint32_t first_realisation;  /* Philox key word 1 of batch element 0 (element r uses first_realisation + r), so
                                    that single realisations of a large ensemble can be stepped on their own */
} orc_problem;

void orc_derive_coeffs(const orc_params* p, double dx, double dy, int32_t prec32,
                       double out[ORC_NCOEF]);

/* One evaluation of the derivative f (the paper's CALCULATE_K) on ONE batch element at time t.
 * psi_* are interleaved complex [ny][nx]; n_* real.  Unused fields may be NULL. */
void orc_derivative(const orc_problem* pb, double t,
                    const double* psi_p, const double* psi_m, const double* n_p, const double* n_m,
                    double* K_p, double* K_m, double* Kn_p, double* Kn_m);

/* n_steps RK4 steps in place on all batch elements; step0 = number of steps already completed
 * (keys the noise and fixes t = step0*dt for the drive).  Returns 0, or 1 on bad arguments. */
int32_t orc_step_rk4(const orc_problem* pb, double* psi_p, double* psi_m, double* n_p, double* n_m,
                     uint64_t step0, int64_t n_steps);

/* ---- adaptive Dormand-Prince 5(4) --------------------------------------------
 * The paper only NAMES the method ("higher-order methods like the RK-Fehlberg or Dormand-Prince can be
 * used for systems requiring adaptive time-stepping"; "adaptive Runge-Kutta methods ... could be
 * optimized within the framework of PHOENIX").  Everything below is DESIGN.md reading Q20:
 *   - tableau: Dormand & Prince, J. Comput. Appl. Math. 6 (1980) 19, the seven-stage 5(4) pair with FSAL,
 *     written out in orc_dp54_tableau; each coefficient is evaluated as a double quotient and, with prec32,
 *     rounded once to float;
 *   - stage s: Y_s = u + h sum_j a_sj K_j, K_s = f(Y_s, t + c_s h); u_new = Y_7 (fifth order);
 *     error estimate E = h sum_j e_j K_j with e = b - b* (b* the embedded fourth-order weights);
 *   - error norm: err = max over all cells, components, reservoirs and batch elements of
 *     |E| / (atol + rtol max(|u|, |u_new|))  (complex modulus for psi, absolute value for n);
 *   - accept iff err <= 1 (or the proposed step is already h_min); step factor q/16 with
 *     q = floor(16 min(4, max(1/4, 0.9 err^(-1/5)))) (q = 64 for err = 0): the QUANTISED factor makes the
 *     step-size sequence an integer sequence that the CUDA path must reproduce bit for bit;
 *     h <- clamp(h_used q/16, h_min, h_max) after every attempt, accepted or not;
 *   - a step that would pass t_end is clipped to land on it exactly; after an accepted clipped step the
 *     unclipped proposal is kept for the next call; the step used is rounded once to float when prec32;
 *   - one step size for the whole batch; noise is not supported (returns 2).
 * Log: one record per ATTEMPT (accepted or rejected): accept flag, q, h used, err. */
typedef struct {
    double atol, rtol;           /* error norm */
    double h_init;               /* first step size tried (used when state->h_next <= 0) */
    double h_min, h_max;         /* clamp of the step size */
    double t_end;                /* integrate until t == t_end */
    int64_t max_attempts;        /* stop after this many attempts of this call even if t < t_end */
} orc_adaptive;

typedef struct {
    double t;                    /* current time (in/out) */
    double h_next;               /* step size the next attempt will try (in/out; <= 0: use h_init) */
    int64_t n_accept, n_reject;  /* counters (in/out) */
} orc_adaptive_state;

/* c[7], a[7][7] (row s, column j < s), b[7] (= a[6][.]), e[7] = b - b*. */
void orc_dp54_tableau(int32_t prec32, double* c, double* a, double* b, double* e);

/* Integrates from st->t to ctl->t_end.  log_* may be NULL; at most log_cap records are written, the
 * number of attempts made is returned in *n_log.  Returns 0; 1 on bad arguments; 2 if noise is on. */
int32_t orc_step_dp54(const orc_problem* pb, double* psi_p, double* psi_m, double* n_p, double* n_m,
                      const orc_adaptive* ctl, orc_adaptive_state* st, int32_t prec32,
                      int32_t* log_accept, int32_t* log_q, double* log_h, double* log_err,
                      int64_t log_cap, int64_t* n_log);

/* Philox4x32-10 (Salmon et al., SC'11): one block. */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* The four 32-bit words drawn for every (realisation, cell) at step `step`:
 * out[batch][ny][nx][4] = Philox(ctr=(cell, step_lo, step_hi, 0), key=(seed, realisation)). */
void orc_noise_u32(int32_t nx, int32_t ny, int32_t batch, uint32_t seed, uint64_t step, uint32_t* out);

/* Map two words to a standard complex normal pair (xi1, xi2) by Box-Muller. */
void orc_normal_pair(uint32_t w0, uint32_t w1, double* xi1, double* xi2);

/* <|psi|^2>(x,y) = (1/batch) sum_r |psi_r|^2 ; psi interleaved complex [batch][ny][nx]. */
void orc_ensemble_mean_density(int32_t nx, int32_t ny, int32_t batch, const double* psi, double* out);

#ifdef __cplusplus
}
#endif
#endif
