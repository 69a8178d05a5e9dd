/*
 * rad_client.c -- the C ABI of include/rad.h used from plain C (no Python, no torch, no CUDA headers):
 * a static particle with a constant acceleration, T steps, state passed in HOST buffers
 * (rad_accumulate_step_host), spectrum returned to HOST memory, compared with the closed form of the
 * rectangle-rule sum (a Dirichlet kernel; pin P2 of tests/test_oracle_pins.py):
 *
 *   S(n, w) = scale w_k^2 (|b|^2 - (n.b)^2) dt^2 sin^2(w T dt / 2) / sin^2(w dt / 2)
 *
 * Build and run (tests/test_abi.py::test_c_client_runs_the_abi_from_plain_c does exactly this):
 *   gcc -std=c11 -I include tests/rad_client.c -L paper_2501_03383_b200 -lrad -lm -o rad_client
 *   LD_LIBRARY_PATH=paper_2501_03383_b200 ./rad_client
 * Exit code 0 and a line "rad_client OK ..." on success.
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "rad.h"

#define ND 3
#define NW 40
#define NP 5 /* one radiating particle + four at rest without acceleration (they add nothing) */

int main(void)
{
    const double dirs[ND][3] = {{1, 0, 0}, {0, 0, 2}, {1, 1, 1}}; /* any length: normalised by the library */
    double omega[NW];
    const double dt = 5e-17, weight = 3.0, b[3] = {2e12, -1e12, 3e12}, r0[3] = {1e-6, -2e-6, 0.5e-6};
    const int T = 23;
    for (int j = 0; j < NW; ++j) omega[j] = 1e14 * pow(1e4, j / (double)(NW - 1));

    rad_config cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.struct_size = sizeof cfg;
    cfg.device = 0;
    cfg.n_dir = ND; cfg.dirs = &dirs[0][0];
    cfg.n_omega = NW; cfg.omega = omega;
    cfg.dt = dt; cfg.t0 = 0.0; cfg.scale = 1.0;
    cfg.state_dtype = RAD_F64;
    rad_handle *h = NULL;
    rad_status st = rad_create(&cfg, &h);
    if (st != RAD_OK) {
        fprintf(stderr, "rad_create: %s: %s\n", rad_status_string(st), rad_last_error(NULL));
        return 2;
    }
    double state[10][NP];
    memset(state, 0, sizeof state);
    for (int c = 0; c < 3; ++c) {
        state[c][0] = r0[c];     /* position */
        state[6 + c][0] = b[c];  /* betadot; beta stays 0 */
        for (int k = 1; k < NP; ++k) state[c][k] = 1e-6 * k;
    }
    for (int k = 0; k < NP; ++k) state[9][k] = weight;
    for (int t = 0; t < T; ++t) {
        st = rad_accumulate_step_host(h, t, NP, state[0], state[1], state[2], state[3], state[4], state[5],
                                      state[6], state[7], state[8], state[9], NULL);
        if (st != RAD_OK) {
            fprintf(stderr, "rad_accumulate_step_host: %s: %s\n", rad_status_string(st), rad_last_error(h));
            return 2;
        }
    }
    double S[ND][NW];
    st = rad_spectrum(h, &S[0][0], RAD_OUT_HOST, NULL);
    if (st != RAD_OK) {
        fprintf(stderr, "rad_spectrum: %s: %s\n", rad_status_string(st), rad_last_error(h));
        return 2;
    }
    double worst = 0.0;
    for (int d = 0; d < ND; ++d) {
        const double nn = sqrt(dirs[d][0] * dirs[d][0] + dirs[d][1] * dirs[d][1] + dirs[d][2] * dirs[d][2]);
        const double nb = (dirs[d][0] * b[0] + dirs[d][1] * b[1] + dirs[d][2] * b[2]) / nn;
        const double amp2 = b[0] * b[0] + b[1] * b[1] + b[2] * b[2] - nb * nb;
        for (int j = 0; j < NW; ++j) {
            const double x = 0.5 * omega[j] * dt, dk = sin(T * x) / sin(x);
            const double ref = weight * weight * amp2 * dt * dt * dk * dk;
            const double peak = weight * weight * amp2 * dt * dt * T * T;
            if (ref >= 1e-6 * peak) worst = fmax(worst, fabs(S[d][j] - ref) / ref);
        }
    }
    printf("rad_client %s: %s, kernel %s, %lld launches, max relative error %.2e\n", worst <= 1e-3 ? "OK" : "FAILED",
           rad_version(), rad_kernel_variant(h), (long long)rad_launch_count(h), worst);
    rad_destroy(h);
    return worst <= 1e-3 ? 0 : 1;
}
