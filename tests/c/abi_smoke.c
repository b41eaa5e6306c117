/*
 * abi_smoke.c -- a plain C caller of libbmlsp2.so: include/bml_sp2.h is the whole interface it needs (no Python, no
 * torch, no C++).  Built by tests/test_boundary.py with gcc, linked against libbmlsp2.so and libcudart.
 *
 *   abi_smoke --no-gpu   argument checks only (every call returns before touching CUDA): runs anywhere
 *   abi_smoke            bml_gershgorin + bml_trace + bml_sp2_dense on a 2 x 2 block-diagonal H of size N = 96 whose
 *                        density matrix has a closed form: each block [[a, b], [b, -a]] contributes the projector
 *                        (I - h / sqrt(a^2 + b^2)) / 2 (Eq. 2 of the paper, with the step function)
 */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <cuda_runtime_api.h>

#include "bml_sp2.h"

#define CHECK(cond) do { if (!(cond)) { printf("FAIL line %d: %s\n", __LINE__, #cond); return 1; } } while (0)

static int no_gpu_checks(void)
{
    bml_sp2_stats_t st;
    bml_matrix_t H = {BML_DENSE, 0, 4, 4, (double *)0x1000, NULL, NULL}, D = H;
    bml_sp2_params_t p = {2, 10, 1e-10, 0.0, 0, 0};
    D.value = (double *)0x2000;
    CHECK(strstr(bml_version(), "sm_100a") != NULL);
    CHECK(strstr(bml_status_string(BML_ERR_ELL_OVERFLOW), "overflow") != NULL);
    CHECK(bml_sp2_dense(NULL, &p, &D, (void *)0x400, 1 << 20, &st, NULL) == BML_ERR_INVALID);
    CHECK(st.status == BML_ERR_INVALID);
    CHECK(bml_sp2_dense(&H, &p, &H, (void *)0x400, 1 << 20, &st, NULL) == BML_ERR_INVALID);        /* D aliases H   */
    p.n_occ = 4;
    CHECK(bml_sp2_dense(&H, &p, &D, (void *)0x400, 1 << 20, &st, NULL) == BML_ERR_INVALID);        /* n_occ == N    */
    p.n_occ = 2;
    CHECK(bml_sp2_dense(&H, &p, &D, (void *)0x400, 16, &st, NULL) == BML_ERR_INVALID);             /* workspace     */
    CHECK(bml_sp2_workspace_bytes(&H, &p) > 2 * 4 * 16 * sizeof(double));
    CHECK(bml_gershgorin(&H, NULL, (void *)0x400, 1024, NULL) == BML_ERR_INVALID);
    CHECK(bml_trace(NULL, (double *)0x400, NULL) == BML_ERR_INVALID);
    bml_sp2_release_cached();                                                                       /* no-op here   */
    printf("OK no-gpu\n");
    return 0;
}

int main(int argc, char **argv)
{
    if (argc > 1 && strcmp(argv[1], "--no-gpu") == 0) return no_gpu_checks();

    enum { N = 96 };
    const size_t bytes = (size_t)N * N * sizeof(double);
    double *h = (double *)calloc((size_t)N * N, sizeof(double)), *d = (double *)malloc(bytes), *ref = (double *)calloc((size_t)N * N, sizeof(double));
    double tr_ref = 0.0;
    for (int q = 0; q < N / 2; ++q) {
        const double a = 0.5 + 0.01 * q, b = 0.3 - 0.002 * q, r = sqrt(a * a + b * b);
        const int i = 2 * q, j = 2 * q + 1;
        h[i * N + i] = a; h[j * N + j] = -a; h[i * N + j] = b; h[j * N + i] = b;
        ref[i * N + i] = 0.5 * (1.0 - a / r); ref[j * N + j] = 0.5 * (1.0 + a / r);
        ref[i * N + j] = ref[j * N + i] = -0.5 * b / r;
        tr_ref += a - a;
    }
    double *dH, *dD, *dS;
    void *ws_raw, *ws;
    CHECK(cudaMalloc((void **)&dH, bytes) == cudaSuccess && cudaMalloc((void **)&dD, bytes) == cudaSuccess &&
          cudaMalloc((void **)&dS, 4 * sizeof(double)) == cudaSuccess);
    CHECK(cudaMemcpy(dH, h, bytes, cudaMemcpyHostToDevice) == cudaSuccess);
    bml_matrix_t H = {BML_DENSE, 0, N, N, dH, NULL, NULL}, D = {BML_DENSE, 0, N, N, dD, NULL, NULL};
    bml_sp2_params_t p = {N / 2, 100, 1e-10, 0.0, 0, 0};
    bml_sp2_stats_t st;
    const size_t wsb = bml_sp2_workspace_bytes(&H, &p);
    CHECK(wsb > 0 && cudaMalloc(&ws_raw, wsb + 1024) == cudaSuccess);
    ws = (void *)(((size_t)ws_raw + 1023) & ~(size_t)1023);           /* the workspace must be 1024-byte aligned */

    double s[4];
    CHECK(bml_gershgorin(&H, dS, ws, wsb, NULL) == BML_OK);
    CHECK(bml_trace(&H, dS + 2, NULL) == BML_OK);
    CHECK(cudaMemcpy(s, dS, 4 * sizeof(double), cudaMemcpyDeviceToHost) == cudaSuccess);
    CHECK(s[0] < -0.5 && s[1] > 0.5 && fabs(s[0] + s[1]) < 1e-12 && fabs(s[2] - tr_ref) < 1e-12);

    const int rc = bml_sp2_dense(&H, &p, &D, ws, wsb, &st, NULL);
    CHECK(rc == BML_OK && st.status == BML_OK && st.n_products == st.m_star + 1 && st.n_products < 40);
    CHECK(st.emin == s[0] && st.emax == s[1]);
    CHECK(cudaMemcpy(d, dD, bytes, cudaMemcpyDeviceToHost) == cudaSuccess);
    double err2 = 0.0, nrm2 = 0.0, tr = 0.0;
    for (int i = 0; i < N * N; ++i) { err2 += (d[i] - ref[i]) * (d[i] - ref[i]); nrm2 += ref[i] * ref[i]; }
    for (int i = 0; i < N; ++i) tr += d[i * N + i];
    CHECK(sqrt(err2 / nrm2) < 1e-10 && fabs(tr - N / 2) < 1e-9);

    /* the fully asynchronous form: stats == NULL, verdict read later */
    bml_sp2_stats_t st2;
    CHECK(bml_sp2_dense(&H, &p, &D, ws, wsb, NULL, NULL) == BML_OK);
    CHECK(bml_sp2_read_stats(ws, &st2, NULL) == BML_OK);
    CHECK(st2.n_products == st.n_products && memcmp(st2.branch, st.branch, sizeof(st.branch)) == 0);
    bml_sp2_release_cached();
    printf("OK gpu products=%d relerr=%.2e\n", st.n_products, sqrt(err2 / nrm2));
    return 0;
}
