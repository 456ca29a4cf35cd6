/* sanitize_main.c -- a stand-alone driver that runs the oracle (bg_oracle.c, compiled into the same program)
 * under AddressSanitizer + UndefinedBehaviorSanitizer ("ASan/UBSan on oracle").
 * TEST INFRASTRUCTURE, like everything under oracle/: built and run by tests/test_oracle_sanitized.py only.
 *
 * The oracle indexes fixed-size thread-local tables with the caller's n and d; every parity verdict rests on it, so
 * one instrumented pass over the extreme shapes pins that it has no out-of-bounds access, no signed overflow, no
 * misaligned or uninitialised-by-construction access.  The buffers here are heap blocks of EXACTLY the documented
 * sizes, so that a read or write one element past an argument array is caught too.
 *
 *   sanitize_main <in> <out>
 *   in:  int32 field, metric; uint32 prime; int32 n, d, batch, states, want_currents; then momenta [batch][n][d]
 *        and polarisations [batch][states][n][d] in the field's input type
 *   out: out [batch][states], currents [batch][states][m][m][d] (if wanted), status [batch], raw
 * Exit code 0, 2 on a usage / IO error, 3 if the oracle rejects the arguments; a sanitizer report aborts
 * (-fno-sanitize-recover=all). */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

int oracle_bg_evaluate(int field, int metric, uint32_t prime, int n, int d, int64_t batch, int states,
                       const void* momenta, const void* polarisations, void* out, void* currents, uint32_t* status);

int main(int argc, char** argv)
{
    if (argc != 3) return 2;
    FILE* f = fopen(argv[1], "rb");
    if (!f) return 2;
    int32_t h[8];
    if (fread(h, sizeof(int32_t), 8, f) != 8) return 2;
    const int field = h[0], metric = h[1], n = h[3], d = h[4], batch = h[5], states = h[6], want_cur = h[7];
    const uint32_t prime = (uint32_t)h[2];
    if (field < 0 || field > 2 || n < 1 || n > 64 || d < 1 || d > 64 || batch < 0 || batch > (1 << 20) || states < 1 ||
        states > 64)
        return 2;
    const size_t in_w = field == 0 ? 4 : 16, out_w = field == 0 ? 4 : field == 1 ? 16 : 2 * sizeof(long double);
    const size_t n_mom = (size_t)batch * n * d, n_pol = n_mom * states, n_out = (size_t)batch * states;
    const size_t n_cur = want_cur ? n_out * (n - 1) * (n - 1) * d : 0;
    void* mom = malloc(n_mom * in_w + (n_mom == 0));
    void* pol = malloc(n_pol * in_w + (n_pol == 0));
    void* out = calloc(n_out + (n_out == 0), out_w);
    void* cur = want_cur ? calloc(n_cur + (n_cur == 0), out_w) : NULL;
    uint32_t* status = calloc((size_t)batch + (batch == 0), 4);
    if (!mom || !pol || !out || !status || (want_cur && !cur)) return 2;
    if (fread(mom, in_w, n_mom, f) != n_mom || fread(pol, in_w, n_pol, f) != n_pol) return 2;
    fclose(f);
    if (oracle_bg_evaluate(field, metric, prime, n, d, batch, states, mom, pol, out, cur, status)) return 3;
    f = fopen(argv[2], "wb");
    if (!f) return 2;
    if (fwrite(out, out_w, n_out, f) != n_out || (want_cur && fwrite(cur, out_w, n_cur, f) != n_cur) ||
        fwrite(status, 4, (size_t)batch, f) != (size_t)batch)
        return 2;
    fclose(f);
    free(mom); free(pol); free(out); free(cur); free(status);
    return 0;
}
