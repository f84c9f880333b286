// Driver of tests/test_oracle_sanitizers.py: the CPU oracle built with -fsanitize=address,undefined and run over every model,
// boundary rule and term on small ragged grids (compute-sanitizer is closed on the GPU pool, so the
// oracle at least is checked for out-of-bounds indexing and undefined behaviour).  Exits 0 when the sanitizers stay quiet.
#include <cmath>
#include <cstdio>
#include <vector>

#include "../oracle/phx_oracle.h"

static double lcg(unsigned long long& s) {
    s = s * 6364136223846793005ull + 1442695040888963407ull;
    return ((double)(s >> 11) / 9007199254740992.0) - 0.5;
}

int main() {
    unsigned long long seed = 12345;
    const int shapes[][3] = {{3, 3, 1}, {8, 5, 2}, {17, 4, 1}, {33, 9, 3}};
    int runs = 0;
    for (const auto& sh : shapes)
        for (int spinor = 0; spinor < 2; ++spinor)
            for (int reservoir = 0; reservoir < 2; ++reservoir)
                for (int bc = 0; bc < 4; ++bc)
                    for (int noise = 0; noise < 2; ++noise) {
                        const int nx = sh[0], ny = sh[1], batch = sh[2];
                        const size_t plane = (size_t)nx * ny, cells = plane * batch;
                        orc_params p = {1.0, 0.5, 1e-2, -2e-3, 2e-2, 0.01, 0.1, 0.15, 0.05, 0.002, 1.0, 0.0, 0.7};
                        orc_problem pb = {};
                        pb.nx = nx; pb.ny = ny; pb.batch = batch; pb.spinor = spinor; pb.reservoir = reservoir; pb.noise = noise;
                        pb.bc_x = bc & 1; pb.bc_y = bc >> 1; pb.seed = 7; pb.first_realisation = 3;
                        orc_derive_coeffs(&p, 0.3, 0.4, (runs & 1), pb.coef);
                        std::vector<double> V(plane), P(plane), E(2 * plane), pp(2 * cells), pm(2 * cells), np_(cells), nm(cells);
                        for (auto& v : V) v = lcg(seed);
                        for (auto& v : P) v = 1.0 + lcg(seed);
                        for (auto& v : E) v = 0.1 * lcg(seed);
                        for (auto& v : pp) v = lcg(seed);
                        for (auto& v : pm) v = lcg(seed);
                        for (auto& v : np_) v = 0.5 + lcg(seed);
                        for (auto& v : nm) v = 0.5 + lcg(seed);
                        pb.V = (runs % 3) ? V.data() : nullptr;
                        pb.P = reservoir ? P.data() : nullptr;
                        pb.E = (runs % 2) ? E.data() : nullptr;
                        if (orc_step_rk4(&pb, pp.data(), spinor ? pm.data() : nullptr, reservoir ? np_.data() : nullptr,
                                         (reservoir && spinor) ? nm.data() : nullptr, 5, 3) != 0) return 2;
                        if (!noise) {
                            orc_adaptive ctl = {1e-6, 1e-6, 0.01, 1e-6, 0.1, 0.05, 50};
                            orc_adaptive_state st = {0.0, 0.0, 0, 0};
                            std::vector<int32_t> la(64), lq(64);
                            std::vector<double> lh(64), le(64);
                            int64_t nlog = 0;
                            if (orc_step_dp54(&pb, pp.data(), spinor ? pm.data() : nullptr, reservoir ? np_.data() : nullptr,
                                              (reservoir && spinor) ? nm.data() : nullptr, &ctl, &st, runs & 1, la.data(), lq.data(),
                                              lh.data(), le.data(), 64, &nlog) != 0) return 3;
                        }
                        for (double v : pp) if (!std::isfinite(v)) return 4;
                        std::vector<double> mean(plane);
                        orc_ensemble_mean_density(nx, ny, batch, pp.data(), mean.data());
                        std::vector<uint32_t> words(cells * 4);
                        orc_noise_u32(nx, ny, batch, 7, 1ull << 33, words.data());
                        ++runs;
                    }
    std::printf("oracle under ASan + UBSan: %d configurations clean\n", runs);
    return 0;
}
