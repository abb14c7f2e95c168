/* Driver for tests/test_oracle_pins2.py::test_P15_oracle_is_clean_under_asan_and_ubsan: a few small runs through
 * every entry point of the oracle, compiled together with oracle/sgp_oracle.c under -fsanitize=address,undefined.
 * Test infrastructure only. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include "sgp_oracle.h"

static unsigned long long s_state = 88172645463325252ULL;
static double urand(void)
{
    s_state ^= s_state << 13; s_state ^= s_state >> 7; s_state ^= s_state << 17;
    return (double)(s_state >> 11) / 9007199254740992.0;
}

#define NY 20
#define NX 16
#define SY 12
#define SX 10
#define CHECK(call) do { int rc_ = (call); if (rc_ != 0) { printf("%s -> %d\n", #call, rc_); return 1; } } while (0)

int main(void)
{
    static oreal psf[2][NY * NX], gS[2][SY * SX], gF[2][NY * NX], truth[NY * NX], f_out[NY * NX], f0[NY * NX];
    unsigned char mask[NY * NX];
    for (int j = 0; j < 2; ++j)
        for (int y = 0; y < NY; ++y)
            for (int x = 0; x < NX; ++x) {
                double dy = y - NY / 2, dx = x - NX / 2, w = 1.2 + 0.5 * j;
                psf[j][y * NX + x] = (oreal)(exp(-(dy * dy + dx * dx) / (2 * w * w)) * (1 + 0.2 * urand()));
            }
    for (int i = 0; i < NY * NX; ++i) { truth[i] = (oreal)(50.0 * urand()); f0[i] = (oreal)(10.0 + urand()); }
    for (int j = 0; j < 2; ++j) {
        for (int i = 0; i < SY * SX; ++i) gS[j][i] = (oreal)floor(30.0 + 20.0 * urand());
        for (int i = 0; i < NY * NX; ++i) gF[j][i] = (oreal)floor(30.0 + 20.0 * urand());
    }
    gF[0][5] = -2;      /* clamped (A17) */
    const oreal *pp[2] = { psf[0], psf[1] }, *gs[2] = { gS[0], gS[1] }, *gf[2] = { gF[0], gF[1] };
    double bc[2] = { 5.0, 6.0 };
    double trJ[64], trA[64], trL[64], trE[64];
    int trR[64], trB[64];
    oracle_options o;
    oracle_result r;

    oracle_options_default(&o); o.max_iter = 25;
    memset(&r, 0, sizeof(r)); r.trace_J = trJ; r.trace_alpha = trA; r.trace_lambda = trL; r.trace_rule = trR; r.trace_backtracks = trB;
    CHECK(oracle_sgp_single(gF[0], psf[0], NULL, 5.0, NULL, f_out, NY, NX, ORACLE_DTYPE, &o, &r));
    CHECK(oracle_rl_single(gF[0], psf[0], gF[1], 0.0, NULL, f_out, NY, NX, ORACLE_DTYPE, &o, &r));
    CHECK(oracle_sgp_multi(2, gf, pp, NULL, bc, NULL, f_out, NY, NX, ORACLE_DTYPE, &o, &r));
    CHECK(oracle_rl_multi(2, gf, pp, NULL, bc, NULL, f_out, NY, NX, ORACLE_DTYPE, &o, &r));
    CHECK(oracle_osem_multi(2, gf, pp, NULL, bc, NULL, f_out, NY, NX, ORACLE_DTYPE, &o, &r));
    o.sigma_R = 1e-3;
    CHECK(oracle_sgp_boundary(2, gs, pp, NULL, bc, 4, 3, SY, SX, NY, NX, NULL, f_out, mask, ORACLE_DTYPE, &o, &r));
    CHECK(oracle_rl_boundary(2, gs, pp, NULL, bc, 4, 3, SY, SX, NY, NX, NULL, f_out, mask, ORACLE_DTYPE, &o, &r));
    CHECK(oracle_osem_boundary(2, gs, pp, NULL, bc, 4, 3, SY, SX, NY, NX, NULL, f_out, mask, ORACLE_DTYPE, &o, &r));

    /* options of round 2: flux constraint, smoothed start, user start, refresh, non-monotone memory, Eq.25 stop */
    o.flux_constraint = 1; o.init = ORACLE_INIT_CONST_SMOOTH; o.init_sigma = 1.5; o.refresh_every = 3; o.armijo_memory = 4;
    CHECK(oracle_sgp_boundary(2, gs, pp, NULL, bc, 4, 3, SY, SX, NY, NX, NULL, f_out, mask, ORACLE_DTYPE, &o, &r));
    o.flux_constraint = 0; o.init = ORACLE_INIT_USER; o.stop_rule = ORACLE_STOP_MINERR;
    r.truth = truth; r.trace_err = trE;
    CHECK(oracle_sgp_multi(2, gf, pp, NULL, bc, f0, f_out, NY, NX, ORACLE_DTYPE, &o, &r));
    CHECK(oracle_rl_multi(2, gf, pp, NULL, bc, f0, f_out, NY, NX, ORACLE_DTYPE, &o, &r));
    CHECK(oracle_osem_multi(2, gf, pp, NULL, bc, f0, f_out, NY, NX, ORACLE_DTYPE, &o, &r));

    /* building blocks */
    static oreal x[9] = { 3, 1, -1, 0.5, 2, 0, 7, -4, 1 }, D[9] = { 1, 1, 1, 2, 0.5, 0, 3, 1, 1 }, y[9];
    double mu;
    CHECK(oracle_project_flux(9, x, D, 4.0, y, &mu));
    static oreal re[15 * 6], im[15 * 6], ore[15 * 6], oim[15 * 6];
    for (int i = 0; i < 90; ++i) { re[i] = (oreal)urand(); im[i] = (oreal)urand(); }
    CHECK(oracle_fft2(15, 6, -1, re, im, ore, oim));
    CHECK(oracle_fft2(15, 6, +1, ore, oim, re, im));
    printf("sanitize-run ok\n");
    return 0;
}
