/*
 * ea_demo.c -- the C ABI of libea_b200.so from plain C (no Python, no torch):
 *   cc ea_demo.c -I ../../include -L .. -lea_b200 -Wl,-rpath,'$ORIGIN/..' -o ea_demo && ./ea_demo
 * L = 8, 64 realizations in two copies, 16 temperatures: thermalize with parallel tempering,
 * measure the overlap of the copies every 10 sweeps, print energy per site, Binder ratio and
 * correlation length by temperature (the observables of the paper's section 5.3).
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include "ea.h"

int main(void)
{
    enum { L = 8, NT = 16, R = 128, N = L * L * L };
    double betas[NT], g[NT], xi[NT];
    int32_t pairs[2][2] = {{0, 2}, {1, 3}};          /* words 0,1 and their copies in words 2,3 */
    static int32_t E[R][NT];
    for (int k = 0; k < NT; ++k) betas[k] = 1.0 / (0.5 * pow(2.0 / 0.5, (double)k / (NT - 1)));

    ea_handle *h = ea_create(L, NT, R, betas, 2024u);
    if (!h) { fprintf(stderr, "ea_create: %s\n", ea_last_error(NULL)); return 1; }
    if (ea_pair_couplings(h) != EA_OK ||                 /* realizations 64.. share the disorder of 0..63 */
        ea_sweep(h, 2000, 1) != EA_OK ||                 /* thermalize, a swap round after every sweep */
        ea_measure_begin(h, &pairs[0][0], 2) != EA_OK ||
        ea_measure(h, 500, 10, 1) != EA_OK ||
        ea_energy(h, &E[0][0]) != EA_OK || ea_get_binder(h, g) != EA_OK ||
        ea_get_correlation_length(h, xi) != EA_OK) {
        fprintf(stderr, "error: %s\n", ea_last_error(h));
        ea_destroy(h);
        return 1;
    }
    printf("%8s %10s %8s %8s\n", "T", "E/N", "Binder", "xi/L");
    for (int t = 0; t < NT; ++t) {
        double e = 0.0;
        for (int r = 0; r < R; ++r) e += E[r][t];
        printf("%8.3f %10.4f %8.4f %8.4f\n", 1.0 / betas[t], e / R / N, g[t], xi[t] / L);
    }
    ea_destroy(h);
    return 0;
}
