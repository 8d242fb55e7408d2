"""the oracle built with -fsanitize=address,undefined runs the worked example (config 1) and a small
batched FP32 tree with every option on (budget, R13 spread, R14 order, kept cells, DFS) and a vector-valued run (R15) without a report, and gives the
golden value. A plain executable, not the ctypes library: ASan wants to be the first thing loaded in its process."""
import os
import subprocess
import tempfile

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

MAIN = r"""
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "zmc_oracle.h"

static void user2_f64(const double* x, int, const double* p, int, double* out, int) { out[0] = p[0] * x[0] * x[0]; out[1] = x[1]; }
static void user2_f32(const float* x, int, const float* p, int, float* out, int) { out[0] = p[0] * x[0] * x[0]; out[1] = x[1]; }

static int run(orc_config& c, int keep, double* value, double* std_) {
    orc_result* r = orc_run(&c, keep);
    if (!r || orc_error(r)) { std::printf("error: %s\n", r ? orc_error(r) : "null"); return 1; }
    orc_get(r, value, std_);
    for (int l = 1; l <= orc_levels(r); ++l) {
        int64_t n = 0, nr = 0, nt = 0;
        orc_level_counts(r, l, &n, &nr, &nt);
        if (keep) {
            std::vector<uint32_t> inst(n), phi(n);
            std::vector<uint64_t> plo(n);
            std::vector<double> mu(n), s(n), tau(n), S(n * c.trials), Q(n * c.trials);
            std::vector<uint8_t> ref(n);
            if (orc_level_cells(r, l, inst.data(), plo.data(), phi.data(), mu.data(), s.data(), tau.data(), ref.data(), S.data()) != n) return 2;
            orc_level_sumsq(r, l, Q.data());
        }
    }
    orc_free(r);
    return 0;
}

int main() {
    double lo3[3] = {0, 0, 0}, up3[3] = {10, 10, 10};
    orc_config c = {};
    c.dim = 3; c.g = 4; c.trials = 5; c.depth = 2; c.n_samples = 2000; c.seed = 1; c.sigma_multiplier = 1.5;
    c.integrand = ORC_SIN_SUM; c.precision = ORC_F64; c.n_instances = 1; c.params_per_instance = 0;
    c.lower = lo3; c.upper = up3; c.params = nullptr;
    double v = 0, s = 0;
    if (run(c, 1, &v, &s)) return 1;
    std::printf("cfg1 %.9f %.9f\n", v, s);
    c.traversal = ORC_DFS;
    double v2 = 0, s2 = 0;
    if (run(c, 0, &v2, &s2)) return 1;
    if (!(v2 - v < 1e-12 && v - v2 < 1e-12)) { std::printf("dfs != bfs\n"); return 3; }   /* same cells, another summation order */

    /* 3 batched 2-D Gaussians in FP32, depth 3, budget 2, spread from the samples, largest-spread order, kept cells */
    double lo2[2] = {0, 0}, up2[2] = {1, 1};
    double p[3][4] = {{1.0, 5.0, 0.5, 0.5}, {1.0, 300.0, 0.3, 0.7}, {2.0, 40.0, 0.2, 0.2}};
    orc_config b = {};
    b.dim = 2; b.g = 3; b.trials = 4; b.depth = 3; b.n_samples = 301; b.seed = 9; b.sigma_multiplier = 0.5;
    b.integrand = ORC_EXP_QUAD; b.precision = ORC_F32; b.n_instances = 3; b.params_per_instance = 4;
    b.lower = lo2; b.upper = up2; b.params = &p[0][0];
    b.max_groups_per_level = 2; b.spread = ORC_SPREAD_SAMPLES; b.budget_order = ORC_BUDGET_LARGEST_SPREAD;
    double bv[3], bs[3];
    if (run(b, 1, bv, bs)) return 1;
    std::printf("batched %.6f %.6f %.6f\n", bv[0], bv[1], bv[2]);
    /* R15: a two-component user integrand in FP32, two instances, depth 3, budget 3, kept cells */
    {
        double pv[2][1] = {{1.0}, {2.0}};
        orc_config v2c = {};
        v2c.dim = 2; v2c.g = 4; v2c.trials = 3; v2c.depth = 3; v2c.n_samples = 77; v2c.seed = 4; v2c.sigma_multiplier = 0.5;
        v2c.precision = ORC_F32; v2c.n_instances = 2; v2c.params_per_instance = 1;
        v2c.lower = lo2; v2c.upper = up2; v2c.params = &pv[0][0]; v2c.max_groups_per_level = 3;
        orc_vec_result* vr = orc_run_vec(&v2c, 2, user2_f64, user2_f32, 1);
        if (!vr || orc_vec_error(vr)) { std::printf("vec error\n"); return 5; }
        double vv[4], vs[4];
        orc_vec_get(vr, vv, vs);
        for (int l = 1; l <= orc_vec_levels(vr); ++l) {
            int64_t n = 0;
            orc_vec_level_counts(vr, l, &n, nullptr, nullptr);
            std::vector<uint32_t> inst(n), phi(n);
            std::vector<uint64_t> plo(n);
            std::vector<double> mu(2 * n), s(2 * n), tau(2 * n), S(2 * n * v2c.trials);
            std::vector<uint8_t> ref(n);
            if (orc_vec_level_cells(vr, l, inst.data(), plo.data(), phi.data(), mu.data(), s.data(), tau.data(), ref.data(), S.data()) != n) return 6;
        }
        std::printf("vec %.6f %.6f %.6f %.6f\n", vv[0], vv[1], vv[2], vv[3]);
        orc_vec_free(vr);
    }
    /* a config the oracle must refuse cleanly */
    b.trials = 300;
    orc_result* r = orc_run(&b, 0);
    if (!r || !orc_error(r)) return 4;
    orc_free(r);
    return 0;
}
"""


def test_oracle_under_asan_ubsan():
    with tempfile.TemporaryDirectory() as d:
        open(os.path.join(d, "main.cpp"), "w").write(MAIN)
        exe = os.path.join(d, "orc_san")
        cmd = ["g++", "-O1", "-g", "-std=c++17", "-ffp-contract=off", "-mfma", "-fsanitize=address,undefined",
               "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-I", os.path.join(ROOT, "oracle"),
               os.path.join(d, "main.cpp"), os.path.join(ROOT, "oracle", "zmc_oracle.cpp"),
               os.path.join(ROOT, "oracle", "zmc_oracle_vec.cpp"), "-o", exe]
        subprocess.run(cmd, check=True)
        env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
        r = subprocess.run([exe], capture_output=True, text=True, env=env)
    assert r.returncode == 0, (r.returncode, r.stdout[-2000:], r.stderr[-4000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
    line = [l for l in r.stdout.splitlines() if l.startswith("cfg1")][0].split()
    # tests/golden/config1_worked.txt: value -4.553120733, std 1.504730423
    assert abs(float(line[1]) - (-4.553120733)) < 2e-9 and abs(float(line[2]) - 1.504730423) < 2e-9
