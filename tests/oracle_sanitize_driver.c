/* Driver for tests/test_oracle_sanitize.py: exercises every entry point of oracle/qmcd_oracle.c
 * (compiled together with it under -fsanitize=address,undefined) on small seeded inputs, including
 * a repeated electron inside one window, a final partial flush, K = 1 and K = n, and the lock-step
 * path.  Exit code 0 and silence from the sanitizers is the pass criterion; the numbers themselves
 * are pinned elsewhere (tests/test_oracle_pins.py).  compute-sanitizer is closed on the GPU pool
 * (DESIGN.md section 4), so this is the memory-safety check the oracle gets. */
#include <stdio.h>
#include <stdlib.h>
#include <math.h>

int orc_slogdet(int n, const double *a, int *sign_out, double *logabs_out);
int orc_inverse(int n, const double *a, double *ainv);
int orc_ratio_bruteforce(int n, const double *A, int j, const double *v, double *R_out);
double orc_sm_ratio(int n, const double *B, int j, const double *v);
int orc_sm_accept(int n, double *B, int j, const double *v);
int orc_run(int path, int batch, int n, int K, int n_moves, int j_begin, double *B, const double *proposals,
            const unsigned char *mask, const double *uniforms, int mode, int final_flush, double *R_out,
            unsigned char *acc_out, int *threads_used);
int orc_run_lockstep(int batch, int n, int K, int n_moves, int j_begin, double *A, double *B,
                     const double *proposals, const unsigned char *mask, const double *uniforms, int mode,
                     int final_flush, double *R_out, unsigned char *acc_out, long *flushes_out, int *threads_used);
int orc_run_jseq(int batch, int n, int K, int n_moves, const int *jseq, int replace, double *B,
                 const double *proposals, const unsigned char *mask, const double *uniforms, int mode,
                 int final_flush, double *R_out, unsigned char *acc_out, long *flushes_out, int *threads_used);
double orc_residual(int n, const double *A, const double *B);

static unsigned long long s_ = 88172645463325252ULL;
static double rnd(void) { s_ ^= s_ << 13; s_ ^= s_ >> 7; s_ ^= s_ << 17; return (double)(s_ >> 11) / 9007199254740992.0 - 0.5; }

int main(void)
{
    const int n = 24, batch = 3, n_moves = 61;
    double *A = malloc(sizeof(double) * batch * n * n), *B = malloc(sizeof(double) * batch * n * n);
    double *B2 = malloc(sizeof(double) * batch * n * n), *A2 = malloc(sizeof(double) * batch * n * n);
    double *P = malloc(sizeof(double) * n_moves * batch * n), *U = malloc(sizeof(double) * n_moves * batch);
    double *R = malloc(sizeof(double) * n_moves * batch);
    unsigned char *mask = malloc(n_moves * batch), *acc = malloc(n_moves * batch);
    int *jseq = malloc(sizeof(int) * n_moves);
    int fail = 0, thr = 0, sign = 0;
    double la = 0.0, Rb = 0.0;
    long fls[3] = {0, 0, 0};
    for (int b = 0; b < batch; ++b) {
        for (int i = 0; i < n * n; ++i) A[(size_t)b * n * n + i] = rnd() / sqrt((double)n);
        for (int i = 0; i < n; ++i) A[(size_t)b * n * n + i * n + i] += 1.0;
        fail |= orc_inverse(n, A + (size_t)b * n * n, B + (size_t)b * n * n) != 0;
    }
    for (int t = 0; t < n_moves; ++t)
        for (int b = 0; b < batch; ++b) {
            const int j = t % n;
            for (int i = 0; i < n; ++i) P[((size_t)t * batch + b) * n + i] = A[(size_t)b * n * n + i * n + j] + 0.3 * rnd() / sqrt((double)n);
            U[t * batch + b] = rnd() + 0.5;
            mask[t * batch + b] = U[t * batch + b] < 0.7;
        }
    for (int t = 0; t < n_moves; ++t) jseq[t] = (t % 5 == 3) ? jseq[t - 2] : (t * 7) % n;   /* repeats inside a window */
    fail |= orc_slogdet(n, A, &sign, &la) != 0;
    fail |= orc_ratio_bruteforce(n, A, 3, P, &Rb) != 0;
    (void)orc_sm_ratio(n, B, 3, P);
    const int Ks[4] = {1, 5, 16, 24};
    for (int path = 1; path <= 2; ++path)
        for (int k = 0; k < 4; ++k)
            for (int mode = 0; mode < 2; ++mode) {
                for (size_t i = 0; i < (size_t)batch * n * n; ++i) B2[i] = B[i];
                fail |= orc_run(path, batch, n, Ks[k], n_moves, 2, B2, P, mask, U, mode, k & 1, R, acc, &thr) != 0;
            }
    for (int k = 0; k < 4; ++k) {
        for (size_t i = 0; i < (size_t)batch * n * n; ++i) { B2[i] = B[i]; A2[i] = A[i]; }
        fail |= orc_run_lockstep(batch, n, Ks[k], n_moves, 0, A2, B2, P, mask, U, 0, 1, R, acc, fls, &thr) != 0;
        for (size_t i = 0; i < (size_t)batch * n * n; ++i) B2[i] = B[i];
        fail |= orc_run_jseq(batch, n, Ks[k], n_moves, jseq, 1, B2, P, mask, U, 0, 1, R, acc, fls, &thr) != 0;
        for (size_t i = 0; i < (size_t)batch * n * n; ++i) B2[i] = B[i];
        fail |= orc_run_jseq(batch, n, Ks[k], n_moves, jseq, 0, B2, P, mask, U, 1, 0, R, acc, fls, &thr) != 0;
    }
    (void)orc_residual(n, A2, B2);
    free(A); free(B); free(B2); free(A2); free(P); free(U); free(R); free(mask); free(acc); free(jseq);
    if (fail) { fprintf(stderr, "oracle call failed\n"); return 1; }
    printf("sanitize driver ok\n");
    return 0;
}
