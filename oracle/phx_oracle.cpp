/*
 * phx_oracle.cpp -- plain, slow, single-threaded CPU ORACLE for the PHOENIX RK4 hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT (see phx_oracle.h).  No code is shared with the CUDA path.
 * Written from /root/reference/PAPER.md; every function cites the passage it follows.
 * Deliberately unfused: K1..K4 and a stage buffer per field, full-grid loop per operation,
 * exactly the structure of Listing 1 and Fig. 2.
 * Build: g++ -O2 -ffp-contract=off (no fast-math, no OpenMP): liboracle.so, the parity oracle, one thread.
 * The "#pragma omp parallel for" lines over the rows / cells of each full-grid loop are ignored by that build; the
 * SAME source compiled with -fopenmp (liboracle_omp.so, oracle/build.py) is the all-host-cores leg of bench.py's
 * cpu_baseline and nothing else.  Every loop iteration writes its own cells only, so
 * the threaded build computes the same bits.
 */
#include "phx_oracle.h"

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstddef>
#include <cstring>
#include <vector>

namespace {

typedef std::complex<double> cplx;

const cplx I_UNIT(0.0, 1.0);

/* i*z and -i*z written out so that no 0*inf products appear. */
inline cplx times_i(const cplx& z) { return cplx(-z.imag(), z.real()); }
inline cplx times_minus_i(const cplx& z) { return cplx(z.imag(), -z.real()); }

double round_to(double v, int32_t prec32) { return prec32 ? (double)(float)v : v; }

/* A field value at integer position (i, j) under the boundary rule of PAPER.md:369:
 * periodic (index taken modulo N) or zero (outside the grid the field is 0). */
struct Grid {
    int nx, ny, bc_x, bc_y;
    template <class T>
    T at(const T* u, int i, int j) const {
        if (i < 0 || i >= nx) {
            if (bc_x) return T(0);
            i = (i % nx + nx) % nx;
        }
        if (j < 0 || j >= ny) {
            if (bc_y) return T(0);
            j = (j % ny + ny) % ny;
        }
        return u[(size_t)j * nx + i];
    }
};

/* The derivative f of PAPER.md:51 for one batch element: K = d(psi)/dt, Kn = dn/dt.
 * Eq. (16) divided through by dt, with Eq. (1) as the scalar case;
 * Listing 2 fixes the sign and form: "+(1/hbar) g |psi|^2 (-i psi)" and
 * "-0.5 gamma psi".  Laplacian: Eq. (8).  Reservoir: Eq. (17).
 * TE-TM: J_pm = Delta_LT (d_x -+ i d_y)^2 acting on psi_-+ (PAPER.md:367-369), discretised with
 * the compact central differences of DESIGN.md reading Q6.  Drive: -(i/hbar) E. */
void derivative(const orc_problem& pb, double t, const cplx* yp, const cplx* ym, const double* np_,
                const double* nm_, cplx* Kp, cplx* Km, double* Knp, double* Knm) {
    const double* c = pb.coef;
    const Grid G = {pb.nx, pb.ny, pb.bc_x, pb.bc_y};
    const cplx drive_phase = std::exp(cplx(0.0, -c[ORC_OMEGA] * t));

    for (int s = 0; s < (pb.spinor ? 2 : 1); ++s) {
        const cplx* y = s == 0 ? yp : ym;          /* this component  psi_sigma   */
        const cplx* yo = s == 0 ? ym : yp;         /* other component psi_-sigma  */
        const double* n = s == 0 ? np_ : nm_;
        cplx* K = s == 0 ? Kp : Km;
        double* Kn = s == 0 ? Knp : Knm;
        const double sign = s == 0 ? -1.0 : +1.0;  /* (d_x - i d_y)^2 in the psi_+ equation */

#pragma omp parallel for schedule(static)
        for (int j = 0; j < pb.ny; ++j) {
            for (int i = 0; i < pb.nx; ++i) {
                const size_t k = (size_t)j * pb.nx + i;
                const cplx yc = y[k];
                const double rho = yc.real() * yc.real() + yc.imag() * yc.imag() - c[ORC_DOFF];
                const double nres = (pb.reservoir && n) ? n[k] : 0.0;

                /* Eq. (8) times hbar/2m:  L = cx (E + W - 2C) + cy (N + S - 2C) */
                const cplx L = c[ORC_CX] * (G.at(y, i + 1, j) + G.at(y, i - 1, j) - 2.0 * yc) +
                               c[ORC_CY] * (G.at(y, i, j + 1) + G.at(y, i, j - 1) - 2.0 * yc);

                double pot = (pb.V ? pb.V[k] : 0.0) + c[ORC_G] * rho + c[ORC_GR] * nres;
                if (pb.spinor) {
                    const cplx oc = yo[k];
                    const double rho_o = oc.real() * oc.real() + oc.imag() * oc.imag() - c[ORC_DOFF];
                    pot += c[ORC_GX] * rho_o;
                }
                const double W = c[ORC_IH] * pot;

                cplx Kc = times_i(L) + times_minus_i(W * yc) + (0.5 * c[ORC_RR] * nres - c[ORC_HGC]) * yc;

                if (pb.spinor) {
                    const cplx oc = yo[k];
                    const cplx Dxx = G.at(yo, i + 1, j) + G.at(yo, i - 1, j) - 2.0 * oc;
                    const cplx Dyy = G.at(yo, i, j + 1) + G.at(yo, i, j - 1) - 2.0 * oc;
                    const cplx Dxy4 = G.at(yo, i + 1, j + 1) - G.at(yo, i + 1, j - 1) -
                                      G.at(yo, i - 1, j + 1) + G.at(yo, i - 1, j - 1);
                    /* (beta/hbar)(d_xx - d_yy -+ 2i d_xy) psi_other */
                    const cplx J = c[ORC_BXX] * Dxx - c[ORC_BYY] * Dyy + sign * c[ORC_BXY] * times_i(Dxy4);
                    Kc += times_minus_i(J);
                }
                if (pb.E) {
                    const cplx Ec(pb.E[2 * k], pb.E[2 * k + 1]);
                    Kc += times_minus_i(c[ORC_IH] * (Ec * drive_phase));
                }
                K[k] = Kc;

                if (pb.reservoir && n) {
                    Kn[k] = (pb.P ? pb.P[k] : 0.0) - (c[ORC_GAMR] + c[ORC_RR] * rho) * nres;
                }
            }
        }
    }
}

/* The paper's INTERMEDIATE_SUM_K (Eq. (9) :208): z = x + alpha*y. */
template <class T>
void two_term_sum(size_t n, const T* x, double alpha, const T* y, T* z) {
#pragma omp parallel for schedule(static)
    for (size_t k = 0; k < n; ++k) z[k] = x[k] + alpha * y[k];
}

/* The paper's FINAL_SUM_K (Eq. (10) :212), weights dt/6, dt/3, dt/3, dt/6. */
template <class T>
void five_term_sum(size_t n, T* x, double a1, const T* y1, double a2, const T* y2, double a3, const T* y3,
                   double a4, const T* y4) {
#pragma omp parallel for schedule(static)
    for (size_t k = 0; k < n; ++k) x[k] = x[k] + a1 * y1[k] + a2 * y2[k] + a3 * y3[k] + a4 * y4[k];
}

/* Philox4x32-10, Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3",
 * SC'11: ten rounds of two 32x32->64 multiplies with key schedule k += (0x9E3779B9, 0xBB67AE85). */
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n1 = (uint32_t)p1;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        const uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* DESIGN.md reading Q13: u = ((w >> 9) + 0.5) * 2^-23 lies in (0,1) and is exactly representable
 * in fp32 (24 significant bits), so both sides start from identical uniforms.  Box-Muller:
 * xi1 + i xi2 = sqrt(-2 ln u1) * exp(2 pi i u2), each a standard normal. */
void normal_pair(uint32_t w0, uint32_t w1, double* xi1, double* xi2) {
    const double two_m23 = 1.0 / 8388608.0;
    const double u1 = ((double)(w0 >> 9) + 0.5) * two_m23;
    const double u2 = ((double)(w1 >> 9) + 0.5) * two_m23;
    const double rad = std::sqrt(-2.0 * std::log(u1));
    const double ang = 2.0 * M_PI * u2;
    *xi1 = rad * std::cos(ang);
    *xi2 = rad * std::sin(ang);
}

}  // namespace

extern "C" {

/* DESIGN.md section 3 "step 0": the canonical coefficient set. */
void orc_derive_coeffs(const orc_params* p, double dx, double dy, int32_t prec32, double out[ORC_NCOEF]) {
    out[ORC_CX] = p->hbar / (2.0 * p->m * dx * dx);   /* (hbar/2m)/dx^2, Eq. (1) x (-i/hbar), Eq. (8) */
    out[ORC_CY] = p->hbar / (2.0 * p->m * dy * dy);
    out[ORC_IH] = 1.0 / p->hbar;
    out[ORC_G] = p->g;
    out[ORC_GX] = p->g_x;
    out[ORC_GR] = p->g_r;
    out[ORC_RR] = p->R;
    out[ORC_HGC] = p->gamma_c / 2.0;
    out[ORC_GAMR] = p->gamma_r;
    out[ORC_BXX] = p->beta / (p->hbar * dx * dx);
    out[ORC_BYY] = p->beta / (p->hbar * dy * dy);
    out[ORC_BXY] = p->beta / (2.0 * p->hbar * dx * dy);
    out[ORC_DT] = p->dt;
    out[ORC_DT6] = p->dt / 6.0;
    out[ORC_DT3] = p->dt / 3.0;
    out[ORC_SIG2] = p->noise_scale * p->dt / (4.0 * dx * dy);   /* Eq. (22) x dt, per real component */
    out[ORC_DOFF] = p->density_offset;
    out[ORC_OMEGA] = p->omega;
    for (int k = 0; k < ORC_NCOEF; ++k) out[k] = round_to(out[k], prec32);
}

void orc_derivative(const orc_problem* pb, double t, const double* psi_p, const double* psi_m,
                    const double* n_p, const double* n_m, double* K_p, double* K_m, double* Kn_p,
                    double* Kn_m) {
    derivative(*pb, t, (const cplx*)psi_p, (const cplx*)psi_m, n_p, n_m, (cplx*)K_p, (cplx*)K_m, Kn_p, Kn_m);
}

/* Eqs. (2)-(6) in the order of Listing 1, on the joint state
 * (psi_+, psi_-, n_+, n_-) (reading Q5), then the noise increment of Eq. (22)
 * added once per step (reading Q12). */
int32_t orc_step_rk4(const orc_problem* pb, double* psi_p_, double* psi_m_, double* n_p_, double* n_m_,
                     uint64_t step0, int64_t n_steps) {
    if (!pb || !psi_p_ || pb->nx < 1 || pb->ny < 1 || pb->batch < 1 || n_steps < 0) return 1;
    if (pb->spinor && !psi_m_) return 1;
    if (pb->reservoir && (!n_p_ || (pb->spinor && !n_m_))) return 1;

    const double* c = pb->coef;
    const size_t N = (size_t)pb->nx * pb->ny;
    const int ncomp = pb->spinor ? 2 : 1;
    const bool res = pb->reservoir != 0;
    const double dt = c[ORC_DT], hdt = 0.5 * c[ORC_DT], dt6 = c[ORC_DT6], dt3 = c[ORC_DT3];

    /* K1..K4 and buffer_wavefunction for every field. */
    std::vector<cplx> K[4][2], buf[2];
    std::vector<double> Kn[4][2], nbuf[2], n_before[2];
    for (int s = 0; s < ncomp; ++s) {
        buf[s].resize(N);
        for (int q = 0; q < 4; ++q) K[q][s].resize(N);
        if (res) {
            nbuf[s].resize(N);
            n_before[s].resize(N);
            for (int q = 0; q < 4; ++q) Kn[q][s].resize(N);
        }
    }

    for (int r = 0; r < pb->batch; ++r) {
        cplx* psi[2] = {(cplx*)psi_p_ + (size_t)r * N, pb->spinor ? (cplx*)psi_m_ + (size_t)r * N : nullptr};
        double* nn[2] = {res ? n_p_ + (size_t)r * N : nullptr, (res && pb->spinor) ? n_m_ + (size_t)r * N : nullptr};

        for (int64_t it = 0; it < n_steps; ++it) {
            const uint64_t step = step0 + (uint64_t)it;
            const double t0 = (double)step * dt;
            const double t_half = ((double)step + 0.5) * dt;
            const double t1 = ((double)step + 1.0) * dt;

            if (res)
                for (int s = 0; s < ncomp; ++s) std::memcpy(n_before[s].data(), nn[s], N * sizeof(double));

            /* CALCULATE_K(1, wavefunction) */
            derivative(*pb, t0, psi[0], psi[1], nn[0], nn[1], K[0][0].data(), K[0][1].data(), Kn[0][0].data(),
                       Kn[0][1].data());
            /* INTERMEDIATE_SUM_K(1, 0.5) */
            for (int s = 0; s < ncomp; ++s) {
                two_term_sum(N, psi[s], hdt, K[0][s].data(), buf[s].data());
                if (res) two_term_sum(N, nn[s], hdt, Kn[0][s].data(), nbuf[s].data());
            }
            /* CALCULATE_K(2, buffer_wavefunction) */
            derivative(*pb, t_half, buf[0].data(), buf[1].data(), nbuf[0].data(), nbuf[1].data(), K[1][0].data(),
                       K[1][1].data(), Kn[1][0].data(), Kn[1][1].data());
            /* INTERMEDIATE_SUM_K(2, 0.5) */
            for (int s = 0; s < ncomp; ++s) {
                two_term_sum(N, psi[s], hdt, K[1][s].data(), buf[s].data());
                if (res) two_term_sum(N, nn[s], hdt, Kn[1][s].data(), nbuf[s].data());
            }
            /* CALCULATE_K(3, buffer_wavefunction) */
            derivative(*pb, t_half, buf[0].data(), buf[1].data(), nbuf[0].data(), nbuf[1].data(), K[2][0].data(),
                       K[2][1].data(), Kn[2][0].data(), Kn[2][1].data());
            /* INTERMEDIATE_SUM_K(3, 1.0) */
            for (int s = 0; s < ncomp; ++s) {
                two_term_sum(N, psi[s], dt, K[2][s].data(), buf[s].data());
                if (res) two_term_sum(N, nn[s], dt, Kn[2][s].data(), nbuf[s].data());
            }
            /* CALCULATE_K(4, buffer_wavefunction) */
            derivative(*pb, t1, buf[0].data(), buf[1].data(), nbuf[0].data(), nbuf[1].data(), K[3][0].data(),
                       K[3][1].data(), Kn[3][0].data(), Kn[3][1].data());
            /* FINAL_SUM_K(4, 1/6, 1/3, 1/3, 1/6) */
            for (int s = 0; s < ncomp; ++s) {
                five_term_sum(N, psi[s], dt6, K[0][s].data(), dt3, K[1][s].data(), dt3, K[2][s].data(), dt6,
                              K[3][s].data());
                if (res)
                    five_term_sum(N, nn[s], dt6, Kn[0][s].data(), dt3, Kn[1][s].data(), dt3, Kn[2][s].data(), dt6,
                                  Kn[3][s].data());
            }

            /* dW of Eq. (22): per real component variance sig2*(gamma_c + R n_t), n_t the reservoir
             * at the start of the step.  Words 0,1 drive psi_+, words 2,3 drive psi_-. */
            if (pb->noise) {
#pragma omp parallel for schedule(static)
                for (size_t k = 0; k < N; ++k) {
                    const uint32_t ctr[4] = {(uint32_t)k, (uint32_t)(step & 0xffffffffu), (uint32_t)(step >> 32), 0u};
                    const uint32_t key[2] = {pb->seed, pb->first_realisation + (uint32_t)r};
                    uint32_t w[4];
                    philox4x32_10(ctr, key, w);
                    for (int s = 0; s < ncomp; ++s) {
                        double xi1, xi2;
                        normal_pair(w[2 * s], w[2 * s + 1], &xi1, &xi2);
                        const double nt = res ? n_before[s][k] : 0.0;
                        const double sigma = std::sqrt(c[ORC_SIG2] * (2.0 * c[ORC_HGC] + c[ORC_RR] * nt));
                        psi[s][k] += sigma * cplx(xi1, xi2);
                    }
                }
            }
        }
    }
    return 0;
}

/* Dormand-Prince 5(4) tableau (J. Comput. Appl. Math. 6 (1980) 19, Table 2), as quotients. */
void orc_dp54_tableau(int32_t prec32, double* c, double* a, double* b, double* e) {
    const double C[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
    const double A[7][7] = {
        {0, 0, 0, 0, 0, 0, 0},
        {1.0 / 5.0, 0, 0, 0, 0, 0, 0},
        {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0, 0},
        {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0, 0},
        {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0, 0},
        {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0, 0},
        {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0, 0}};
    /* embedded fourth-order weights b* */
    const double BS[7] = {5179.0 / 57600.0, 0.0, 7571.0 / 16695.0, 393.0 / 640.0, -92097.0 / 339200.0,
                          187.0 / 2100.0, 1.0 / 40.0};
    for (int s = 0; s < 7; ++s) {
        c[s] = round_to(C[s], prec32);
        for (int j = 0; j < 7; ++j) a[7 * s + j] = round_to(A[s][j], prec32);
        b[s] = round_to(A[6][s], prec32);
        e[s] = round_to(A[6][s] - BS[s], prec32);
    }
}

int32_t orc_step_dp54(const orc_problem* pb, double* psi_p_, double* psi_m_, double* n_p_, double* n_m_,
                      const orc_adaptive* ctl, orc_adaptive_state* st, int32_t prec32,
                      int32_t* log_accept, int32_t* log_q, double* log_h, double* log_err,
                      int64_t log_cap, int64_t* n_log) {
    if (!pb || !psi_p_ || !ctl || !st || pb->nx < 1 || pb->ny < 1 || pb->batch < 1) return 1;
    if (pb->spinor && !psi_m_) return 1;
    if (pb->reservoir && (!n_p_ || (pb->spinor && !n_m_))) return 1;
    if (!(ctl->atol >= 0) || !(ctl->rtol >= 0) || !(ctl->atol + ctl->rtol > 0) || !(ctl->h_min > 0) ||
        !(ctl->h_max >= ctl->h_min))
        return 1;
    if (pb->noise) return 2;

    const size_t N = (size_t)pb->nx * pb->ny;
    const int ncomp = pb->spinor ? 2 : 1;
    const bool res = pb->reservoir != 0;
    const int B = pb->batch;
    double c[7], a[49], b[7], e[7];
    orc_dp54_tableau(prec32, c, a, b, e);

    /* per batch element and field: K_1..K_7, the stage input Y and the candidate u_new */
    std::vector<cplx> K[7][2], Y[2], Un[2];
    std::vector<double> Kn[7][2], Yn[2], Unn[2];
    for (int s = 0; s < ncomp; ++s) {
        Y[s].resize(N * B);
        Un[s].resize(N * B);
        for (int q = 0; q < 7; ++q) K[q][s].resize(N * B);
        if (res) {
            Yn[s].resize(N * B);
            Unn[s].resize(N * B);
            for (int q = 0; q < 7; ++q) Kn[q][s].resize(N * B);
        }
    }
    cplx* psi[2] = {(cplx*)psi_p_, pb->spinor ? (cplx*)psi_m_ : nullptr};
    double* nn[2] = {res ? n_p_ : nullptr, (res && pb->spinor) ? n_m_ : nullptr};

    /* f on every batch element */
    auto f_all = [&](double t, cplx* const y[2], double* const yn[2], int q) {
        for (int r = 0; r < B; ++r) {
            const size_t o = (size_t)r * N;
            derivative(*pb, t, y[0] + o, y[1] ? y[1] + o : nullptr, yn[0] ? yn[0] + o : nullptr,
                       yn[1] ? yn[1] + o : nullptr, K[q][0].data() + o, ncomp == 2 ? K[q][1].data() + o : nullptr,
                       res ? Kn[q][0].data() + o : nullptr, (res && ncomp == 2) ? Kn[q][1].data() + o : nullptr);
        }
    };

    double t = st->t;
    double h = st->h_next > 0 ? st->h_next : ctl->h_init;
    if (h < ctl->h_min) h = ctl->h_min;
    if (h > ctl->h_max) h = ctl->h_max;
    bool have_k1 = false;                 /* FSAL: K_1 of this attempt is K_7 of the last accepted one */
    int64_t attempts = 0;
    while (t < ctl->t_end && attempts < ctl->max_attempts) {
        /* the step actually taken: clipped so that the call lands on t_end; rounded once to T */
        const bool clipped = t + h >= ctl->t_end;
        const double hu = round_to(clipped ? ctl->t_end - t : h, prec32);

        if (!have_k1) {
            f_all(t, psi, nn, 0);
            have_k1 = true;
        }
        /* stages 2..7: Y_s = u + hu sum_j a_sj K_j, K_s = f(Y_s, t + c_s hu); Y_7 is u_new */
        for (int s = 1; s < 7; ++s) {
            for (int comp = 0; comp < ncomp; ++comp) {
                cplx* dst = s == 6 ? Un[comp].data() : Y[comp].data();
                for (size_t k = 0; k < N * B; ++k) {
                    cplx acc(0.0, 0.0);
                    for (int j = 0; j < s; ++j) acc += a[7 * s + j] * K[j][comp][k];
                    dst[k] = psi[comp][k] + hu * acc;
                }
                if (res) {
                    double* dn = s == 6 ? Unn[comp].data() : Yn[comp].data();
                    for (size_t k = 0; k < N * B; ++k) {
                        double acc = 0.0;
                        for (int j = 0; j < s; ++j) acc += a[7 * s + j] * Kn[j][comp][k];
                        dn[k] = nn[comp][k] + hu * acc;
                    }
                }
            }
            cplx* const ys[2] = {s == 6 ? Un[0].data() : Y[0].data(),
                                 ncomp == 2 ? (s == 6 ? Un[1].data() : Y[1].data()) : nullptr};
            double* const yns[2] = {res ? (s == 6 ? Unn[0].data() : Yn[0].data()) : nullptr,
                                    (res && ncomp == 2) ? (s == 6 ? Unn[1].data() : Yn[1].data()) : nullptr};
            f_all(t + c[s] * hu, ys, yns, s);
        }
        /* error norm */
        double err = 0.0;
        for (int comp = 0; comp < ncomp; ++comp) {
            for (size_t k = 0; k < N * B; ++k) {
                cplx E(0.0, 0.0);
                for (int j = 0; j < 7; ++j) E += e[j] * K[j][comp][k];
                const double sc = ctl->atol + ctl->rtol * std::max(std::abs(psi[comp][k]), std::abs(Un[comp][k]));
                err = std::max(err, std::abs(hu * E) / sc);
            }
            if (res)
                for (size_t k = 0; k < N * B; ++k) {
                    double E = 0.0;
                    for (int j = 0; j < 7; ++j) E += e[j] * Kn[j][comp][k];
                    const double sc = ctl->atol + ctl->rtol * std::max(std::fabs(nn[comp][k]), std::fabs(Unn[comp][k]));
                    err = std::max(err, std::fabs(hu * E) / sc);
                }
        }
        /* controller */
        const bool accept = err <= 1.0 || h <= ctl->h_min;       /* a proposal that cannot shrink is taken as it is */
        double fac = err > 0.0 ? 0.9 * std::pow(err, -0.2) : 4.0;
        fac = std::min(4.0, std::max(0.25, fac));
        const int32_t q = (int32_t)std::floor(16.0 * fac);
        if (attempts < log_cap) {
            if (log_accept) log_accept[attempts] = accept ? 1 : 0;
            if (log_q) log_q[attempts] = q;
            if (log_h) log_h[attempts] = hu;
            if (log_err) log_err[attempts] = err;
        }
        ++attempts;
        if (accept) {
            for (int comp = 0; comp < ncomp; ++comp) {
                std::memcpy(psi[comp], Un[comp].data(), N * B * sizeof(cplx));
                K[0][comp].swap(K[6][comp]);                      /* FSAL */
                if (res) {
                    std::memcpy(nn[comp], Unn[comp].data(), N * B * sizeof(double));
                    Kn[0][comp].swap(Kn[6][comp]);
                }
            }
            t = clipped ? ctl->t_end : t + hu;
            ++st->n_accept;
            /* (a clipped step says nothing about the step size the dynamics allow: the proposal h is kept) */
            if (!clipped) h = std::min(ctl->h_max, std::max(ctl->h_min, hu * (double)q / 16.0));
        } else {
            ++st->n_reject;
            h = std::min(ctl->h_max, std::max(ctl->h_min, hu * (double)q / 16.0));
        }
    }
    st->t = t;
    st->h_next = h;
    if (n_log) *n_log = attempts;
    return 0;
}

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox4x32_10(ctr, key, out);
}

void orc_noise_u32(int32_t nx, int32_t ny, int32_t batch, uint32_t seed, uint64_t step, uint32_t* out) {
    const size_t N = (size_t)nx * ny;
    for (int r = 0; r < batch; ++r)
        for (size_t k = 0; k < N; ++k) {
            const uint32_t ctr[4] = {(uint32_t)k, (uint32_t)(step & 0xffffffffu), (uint32_t)(step >> 32), 0u};
            const uint32_t key[2] = {seed, (uint32_t)r};
            philox4x32_10(ctr, key, out + 4 * ((size_t)r * N + k));
        }
}

void orc_normal_pair(uint32_t w0, uint32_t w1, double* xi1, double* xi2) { normal_pair(w0, w1, xi1, xi2); }

/* ensemble average over the Monte-Carlo realisations, plain sum over r. */
void orc_ensemble_mean_density(int32_t nx, int32_t ny, int32_t batch, const double* psi, double* out) {
    const size_t N = (size_t)nx * ny;
    for (size_t k = 0; k < N; ++k) {
        double acc = 0.0;
        for (int r = 0; r < batch; ++r) {
            const double re = psi[2 * ((size_t)r * N + k)], im = psi[2 * ((size_t)r * N + k) + 1];
            acc += re * re + im * im;
        }
        out[k] = acc / (double)batch;
    }
}

}  // extern "C"
