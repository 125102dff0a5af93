// Host-only driver for the ASan/UBSan job (tests/test_sanitizers.py): exercises the plain-C oracle
// (oracle/lipfit_oracle.c) and the host LBFGS of the product (csrc/lbfgs.cpp, step a5) on small inputs,
// including ragged sizes, zero weights, duplicates and infinite region thresholds.  Built with
//   g++ -fsanitize=address,undefined -fno-sanitize-recover=all
// so any out-of-bounds access, use of uninitialised stack, signed overflow or misaligned access aborts.
// The two code bases are only linked into this TEST binary side by side; neither calls the other:
// LBFGS is driven by a Rosenbrock function defined here.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <vector>

#include "../oracle/lipfit_oracle.h"
#include "../paper_2606_04670_b200/csrc/lbfgs.h"

static uint64_t rng_state = 0x9E3779B97F4A7C15ull;
static double rnd() {  // splitmix64 -> [0, 1)
    uint64_t z = (rng_state += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    return static_cast<double>(z >> 11) / 9007199254740992.0;
}

#define CHECK(cond)                                                        \
    do {                                                                   \
        if (!(cond)) {                                                     \
            std::fprintf(stderr, "CHECK failed: %s (line %d)\n", #cond, __LINE__); \
            return 1;                                                      \
        }                                                                  \
    } while (0)

int main() {
    for (int d : {1, 3, 8, 17}) {
        const int64_t N = 97, Q = 53;
        std::vector<float> X(N * d), Xq(Q * d), y(N), w(d);
        std::vector<int32_t> mask(d), mon(d);
        std::vector<float> a(d), b(d);
        for (auto& v : X) v = static_cast<float>(rnd());
        for (auto& v : Xq) v = static_cast<float>(rnd());
        for (auto& v : y) v = static_cast<float>(rnd());
        for (int i = 0; i < d; ++i) {
            w[i] = (i % 4 == 3) ? 0.f : static_cast<float>(0.5 + rnd());
            mask[i] = i % 3 - 1;
            mon[i] = i % 5;
            a[i] = (i % 7 == 1) ? -INFINITY : 0.3f;
            b[i] = (i % 7 == 2) ? INFINITY : 0.6f;
        }
        for (int j = 0; j < d; ++j) X[(N - 1) * d + j] = X[j];  // a duplicate datum
        std::vector<double> U(Q), L(Q), G(Q);
        for (int norm = 1; norm <= 3; ++norm) {
            CHECK(oracle_bounds(X.data(), y.data(), N, d, Xq.data(), Q, 1.5, mask.data(), norm, w.data(), U.data(),
                                L.data(), G.data()) == 0);
            CHECK(oracle_bounds(X.data(), y.data(), N, d, Xq.data(), 0, 1.5, nullptr, norm, nullptr, nullptr,
                                nullptr, nullptr) == 0);
            CHECK(oracle_bounds_region(X.data(), y.data(), N, d, Xq.data(), Q, 1.5, mon.data(), a.data(), b.data(),
                                       norm, w.data(), U.data(), L.data(), G.data()) == 0);
            const float wk[3] = {0.5f, 0.3f, 0.2f};
            CHECK(oracle_bounds_topk(X.data(), y.data(), N, d, Xq.data(), Q, 1.5, mask.data(), norm, w.data(), 3, wk,
                                     U.data(), L.data(), G.data()) == 0);
            const int k = 7;
            std::vector<int32_t> idx(Q * k);
            std::vector<double> dist(Q * k);
            for (int side = -1; side <= 1; ++side)
                CHECK(oracle_knn(X.data(), N, d, Xq.data(), Q, mask.data(), side, norm, w.data(), k, idx.data(),
                                 dist.data()) == 0);
            std::vector<double> eps(N, 0.01), grad(N);
            double F = 0, mv = 0;
            CHECK(oracle_smooth_objective(X.data(), y.data(), N, d, 0.2, mask.data(), norm, w.data(), 1.0, eps.data(),
                                          &F, grad.data()) == 0);
            CHECK(std::isfinite(F));
            CHECK(oracle_max_violation(X.data(), y.data(), N, d, 0.2, mask.data(), norm, w.data(), eps.data(), &mv) == 0);
            double Lc = 0;
            CHECK(oracle_lipschitz_constant(X.data(), y.data(), N, d, nullptr, norm, w.data(), &Lc) == 0);
            const int J = 16, S = 300;
            std::vector<int32_t> pi(S), pk(S);
            for (int s = 0; s < S; ++s) {
                pi[s] = static_cast<int32_t>(rnd() * N) % N;
                pk[s] = static_cast<int32_t>(rnd() * N) % N;
            }
            std::vector<double> knots(J), table(N * J), rows_out(3 * J);
            CHECK(oracle_distance_quantiles(X.data(), N, d, norm, w.data(), pi.data(), pk.data(), S, J, knots.data()) == 0);
            CHECK(oracle_local_lipschitz(X.data(), y.data(), N, d, norm, w.data(), knots.data(), J, table.data()) == 0);
            const int64_t rows[3] = {0, N - 1, 5};
            CHECK(oracle_local_lipschitz_rows(X.data(), y.data(), N, d, norm, w.data(), knots.data(), J, rows, 3,
                                              rows_out.data()) == 0);
            for (int j = 0; j < J; ++j) CHECK(rows_out[2 * J + j] == table[5 * J + j]);
            CHECK(oracle_values_local(X.data(), y.data(), N, d, Xq.data(), Q, norm, w.data(), knots.data(), J,
                                      table.data(), U.data(), L.data(), G.data()) == 0);
        }
        // bad arguments return codes, never touch memory
        CHECK(oracle_bounds(nullptr, y.data(), N, d, Xq.data(), Q, 1.0, nullptr, 2, nullptr, U.data(), L.data(),
                            G.data()) != 0);
        CHECK(oracle_bounds(X.data(), y.data(), N, d, Xq.data(), Q, -1.0, nullptr, 2, nullptr, U.data(), L.data(),
                            G.data()) != 0);
    }
    // ---- host LBFGS (csrc/lbfgs.cpp): Rosenbrock in n = 10, history 5 and 20, and an evaluation error ----
    for (int history : {1, 5, 20}) {
        const int n = 10;
        std::vector<double> x(n, -1.2);
        lipfit::LbfgsResult res;
        int accepted = -1;
        int rc = lipfit::lbfgs_minimize(
            n, x.data(),
            [&](const double* v, double* f, double* g) {
                double s = 0;
                for (int i = 0; i < n; ++i) g[i] = 0;
                for (int i = 0; i + 1 < n; ++i) {
                    const double t1 = v[i + 1] - v[i] * v[i], t2 = 1 - v[i];
                    s += 100 * t1 * t1 + t2 * t2;
                    g[i] += -400 * v[i] * t1 - 2 * t2;
                    g[i + 1] += 200 * t1;
                }
                *f = s;
                return 0;
            },
            2000, 1e-9, history, &res, [&](int e) { accepted = e; });
        CHECK(rc == 0);
        CHECK(res.f <= res.f0);
        CHECK(accepted >= 0 && accepted < res.evals);
        if (history >= 5) {
            for (int i = 0; i < n; ++i) CHECK(std::fabs(x[i] - 1.0) < 1e-5);
        }
    }
    {
        std::vector<double> x(4, 0.5);
        lipfit::LbfgsResult res;
        int calls = 0;
        int rc = lipfit::lbfgs_minimize(
            4, x.data(),
            [&](const double* v, double* f, double* g) {
                if (++calls == 3) return -5;
                *f = 0;
                for (int i = 0; i < 4; ++i) {
                    *f += v[i] * v[i] * v[i] * v[i];
                    g[i] = 4 * v[i] * v[i] * v[i];
                }
                return 0;
            },
            50, 1e-12, 20, &res);
        CHECK(rc == -5);
    }
    std::puts("sanitize_driver ok");
    return 0;
}
