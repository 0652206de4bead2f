// sanitize_main.cpp — drives every entry point of the oracle on small inputs; built by tests/test_oracle_sanitize.py
// with -fsanitize=address,undefined.  TEST INFRASTRUCTURE, like everything under oracle/.
#include <cmath>
#include <cstdio>
#include <vector>

#include "ens_oracle.cpp"

int main() {
    int bad = 0;
    for (int n = 2; n <= 16; n += (n < 6 ? 1 : 5)) {
        const int64_t n_sys = 5;
        std::vector<double> pos(n_sys * n * 3, 0.0), vel(n_sys * n * 3, 0.0), mass(n_sys * n, 1e-4), time(n_sys, 0.0);
        std::vector<int32_t> status(n_sys, 0);
        std::vector<int64_t> nsteps(n_sys, 0), nrej(n_sys, 0);
        for (int64_t s = 0; s < n_sys; ++s) {
            mass[s * n] = 1.0;
            for (int i = 1; i < n; ++i) {  // circular, coplanar, spaced by 1.4, phases spread by system
                const double a = std::pow(1.4, i - 1), ph = 0.7 * i + 0.3 * s;
                pos[(s * n + i) * 3 + 0] = a * std::cos(ph);
                pos[(s * n + i) * 3 + 1] = a * std::sin(ph);
                vel[(s * n + i) * 3 + 0] = -std::sin(ph) / std::sqrt(a);
                vel[(s * n + i) * 3 + 1] = std::cos(ph) / std::sqrt(a);
            }
        }
        const double dts[7] = {0.01, 0.05, 0.02, 0.01, 0.01, 0.05, 0.02};
        for (int integ = 0; integ <= 6; ++integ) {
            for (int prec = 0; prec <= 1; ++prec) {
                std::vector<double> p = pos, v = vel, t = time;
                std::vector<int32_t> st = status;
                std::vector<int64_t> ns = nsteps, nr = nrej;
                const int rc = orc_integrate2(integ, n_sys, n, p.data(), v.data(), mass.data(), t.data(), st.data(), ns.data(),
                                              dts[integ], 1.0, 40, 0.01, 100.0, prec, 2, 1e-8, nr.data());
                for (double q : p) bad += !std::isfinite(q);
                bad += rc != 0;
            }
        }
        std::vector<double> E(n_sys), L(3 * n_sys), a(3 * n), j(3 * n), ex(3 * n), ev(3 * n);
        bad += orc_energy(n_sys, n, pos.data(), vel.data(), mass.data(), E.data(), L.data(), 1) != 0;
        bad += orc_acc_jerk(n, pos.data(), vel.data(), mass.data(), a.data(), j.data(), 0) != 0;
        std::vector<double> x(pos.begin(), pos.begin() + 3 * n), w(vel.begin(), vel.begin() + 3 * n);
        bad += orc_hermite_step(n, x.data(), w.data(), mass.data(), 0.01, 2, 1) != 0;
        bad += orc_rkck_step(n, x.data(), w.data(), mass.data(), 0.01, ex.data(), ev.data(), 0) != 0;
        double h = 0.5, r = 0.0, dt = 0.0;
        int ok = 0;
        bad += orc_rkck_adaptive_trial(n, x.data(), w.data(), mass.data(), &h, 1e-9, &r, &ok, 0) != 0;
        bad += orc_adaptive_dt(n, x.data(), w.data(), mass.data(), 0.02, &dt, 0) != 0;
        std::vector<double> Q(3 * n), V(3 * n), x2(3 * n), v2(3 * n);
        bad += orc_dh_roundtrip(n, x.data(), w.data(), mass.data(), Q.data(), V.data(), x2.data(), v2.data()) != 0;
    }
    double c[4], q[3] = {1.0, 0.2, -0.1}, p[3] = {0.3, 1.1, 0.2};
    for (double z : {-30.0, -0.05, 0.0, 0.09, 3.0, 200.0}) bad += orc_stumpff(z, c, 0) != 0;
    int it = 0;
    for (double tau : {0.05, 3.0, -11.0, 40.0}) bad += orc_kepler_drift(q, p, 1.0, tau, 0, &it) != 0;  // includes the fallback
    double tc[6], ta[30], tb5[6], tb4[6];
    bad += orc_rkck_tableau(tc, ta, tb5, tb4) != 0;
    std::printf("oracle sanitize run: %d problems\n", bad);
    return bad ? 1 : 0;
}
