/*
 * bml_graph.h -- C ABI of libbmlsp2.so, part 3: the graph-based density-matrix construction of arxiv 2401.13772
 * section VIII.B (Eq. 15, Listing 11) on one B200, sparse ELLPACK-R in, sparse ELLPACK-R out.
 *
 *   A_ij = 1 if |H_ij| >= graph_tol and i != j                                 Eq. 15; the graph is H's own
 *   pi_k^ch = pi_k^c  U  { o : A_lo = 1 for some l in pi_k^c }                 core-halo parts
 *   h^k = H[pi_k^ch, pi_k^ch]   dense                                          bml_matrix2submatrix
 *   d^k = f_mu(h^k)             the local solver: bml_chebyshev.h
 *   D[l, :] <- d^k[l, :]        for the core nodes l of part k                 bml_submatrix2matrix
 *
 * The core partition is an INPUT (graph partitioning is external: METIS etc.).  Everything else runs in the
 * library's kernels: halo construction, gather, one Chebyshev expansion per part (each on its own Gershgorin
 * interval; parts of equal size are expanded as one batch whose products share grouped launches, otherwise parts run
 * back to back with the whole GPU each), thresholded scatter of the core rows.
 * Readings of the paper fixed by this interface: DESIGN.md "Readings" G1-G6.  Conventions as in bml_sp2.h.
 */
#ifndef BML_GRAPH_H
#define BML_GRAPH_H

#include "bml_chebyshev.h"

#ifdef __cplusplus
extern "C" {
#endif

#define BML_GRAPH_MAX_PARTS 256
#define BML_ERR_PART_CAPACITY (-7)   /* a core+halo part is larger than params.part_capacity; stats->max_part_size says by how much */

typedef struct {
    double  mu, beta;       /* local solver (bml_cheb_params_t): chemical potential, 1 / (k_B T)                   */
    double  graph_tol;      /* tau of Eq. 15: o is a neighbour of l iff |H_lo| >= graph_tol, o != l                */
    double  drop_tol;       /* D keeps |v| >= drop_tol or the diagonal (the SP2 path's rule); 0 keeps everything   */
    int32_t k, m;           /* local solver: Eq. 10 factors, L + 1 = k m                                            */
    int32_t n_parts;        /* 1 .. BML_GRAPH_MAX_PARTS                                                             */
    int32_t part_capacity;  /* largest core+halo size the workspace is provisioned for (<= N)                       */
} bml_graph_params_t;

/* Filled on the HOST when bml_graph_chebyshev_ellpack returns. */
typedef struct {
    int32_t status;         /* = return value                                                                       */
    int32_t n_parts;
    int32_t overflow_row;   /* status -3: lowest row of D needing more than D->M slots, else -1                     */
    int32_t max_part_size;  /* largest core+halo size found                                                         */
    int32_t n_products;     /* matrix products executed, all parts                                                  */
    int32_t pad;
    int32_t part_size[BML_GRAPH_MAX_PARTS];   /* core+halo nodes of part k                                          */
    int32_t core_size[BML_GRAPH_MAX_PARTS];   /* core nodes of part k                                               */
} bml_graph_stats_t;

/*
 * D <- rows of f_mu(h^k) for the core nodes of every part (Listing 11 with the Chebyshev local solver).
 * H: ELLPACK-R, symmetric, rows in any order.  D: ELLPACK-R, same N, its OWN row capacity D->M (rows of D are as long
 * as the core+halo part unless drop_tol cuts them), rows written in ascending column order, unused slots (0.0, 0).
 * d_core_offsets: DEVICE int32[n_parts + 1], d_core_nodes: DEVICE int32[N]: part k owns
 *   d_core_nodes[d_core_offsets[k] .. d_core_offsets[k+1]); every node in exactly one part (not checked).
 * d_workspace >= bml_graph_workspace_bytes(N, n_parts, part_capacity, k, m), 1024-byte aligned.
 * One host synchronisation after the halo pass (the part sizes decide the launch shapes) and one at the end.
 * Returns 0, -1, -2 (a part with e_max = e_min), -3, -4, -7.
 */
BML_API size_t bml_graph_workspace_bytes(int64_t N, int32_t n_parts, int32_t part_capacity, int32_t k, int32_t m);
BML_API int bml_graph_chebyshev_ellpack(const bml_matrix_t *H, const int32_t *d_core_offsets, const int32_t *d_core_nodes,
                                        const bml_graph_params_t *p, bml_matrix_t *D, void *d_workspace,
                                        size_t workspace_bytes, bml_graph_stats_t *stats, void *cuda_stream);

/*
 * The three data-movement steps, exported for per-kernel parity tests and timing.  All asynchronous; return 0, -1, -4.
 *
 * bml_graph_core_halo: for every part, the ascending node list of pi_k^ch and the flag "is a core node".
 *   d_part_nodes: DEVICE int32[n_parts * N], d_is_core: DEVICE uint8[n_parts * N] (row k holds part k, entries beyond
 *   its size untouched), d_part_sizes: DEVICE int32[2 * n_parts] <- { core+halo size, core size } per part.
 *   d_workspace: DEVICE scratch of n_parts * N bytes.
 * bml_matrix2submatrix_ellpack: h[a * ld + b] <- H[nodes[a], nodes[b]] (0 where H stores nothing), a, b < s;
 *   d_nodes ascending.  Every stored entry is taken (no threshold).
 * bml_submatrix2matrix_ellpack: for every a with d_is_core[a]: row nodes[a] of D <- { (nodes[b], d[a * ld + b]) :
 *   |d| >= drop_tol or nodes[b] == nodes[a] }, ascending; nnz set; unused slots (0.0, 0).  A row that needs more than
 *   D->M slots is left untouched and atomicMin'ed into *d_overflow_row (the caller initialises it to INT32_MAX).
 */
BML_API int bml_graph_core_halo(const bml_matrix_t *H, const int32_t *d_core_offsets, const int32_t *d_core_nodes,
                                int32_t n_parts, double graph_tol, int32_t *d_part_nodes, uint8_t *d_is_core,
                                int32_t *d_part_sizes, void *d_workspace, size_t workspace_bytes, void *cuda_stream);
BML_API int bml_matrix2submatrix_ellpack(const bml_matrix_t *H, const int32_t *d_nodes, int32_t s, double *d_h, int64_t ld,
                                         void *cuda_stream);
BML_API int bml_submatrix2matrix_ellpack(const double *d_d, int64_t ld, const int32_t *d_nodes, const uint8_t *d_is_core,
                                         int32_t s, double drop_tol, bml_matrix_t *D, int32_t *d_overflow_row,
                                         void *cuda_stream);

/*
 * Listing 11 with SP2 (section IV.A, Eq. 5-7) as the local solver `prg_build_DM`.  The graph theory of the
 * method applies the SAME matrix function to every part, and SP2's function is fixed by its spectral bounds
 * and its branch sequence, so all parts share one SP2 polynomial (reading G3'):
 *   X_0^k = (e_max I - h^k) / (e_max - e_min)     with the Gershgorin bounds of the WHOLE H (bml_gershgorin), Eq. 5
 *   b_m = [ t_m - n_occ <= 0 ],  t_m = sum_k sum_{a in core of k} (X_m^k)_aa          one branch bit, Eq. 6-7
 *   e_m = sqrt(sum_k ||(X_m^k)^2 - X_m^k||_F^2) / sqrt(sum_k ||X_m^k||_F^2)           one stop test, rules S1-S3
 *   D[l, :] <- X_{m*}^k[l, :] for the core nodes l of part k.
 * A product of ALL parts is one persistent launch over the parts' upper-triangle tiles (parts may differ in size); the
 * branch bit and the stop test stay on the device as in bml_sp2_dense.  One host synchronisation after the halo pass
 * (part sizes decide buffer offsets) and one at the end.  n_parts <= BML_GRAPH_MAX_PARTS.
 * d_workspace >= bml_graph_sp2_workspace_bytes(N, n_parts, part_capacity), 1024-byte aligned.
 * Returns the SP2 status (0, 1, 2) or -1, -2, -3 (a row of D needs more than D->M slots), -4, -7.
 */
typedef struct {
    double  graph_tol;      /* tau of Eq. 15                                                                        */
    double  drop_tol;       /* D keeps |v| >= drop_tol or the diagonal                                              */
    double  idem_tol;       /* tolerance on e_m                                                                     */
    int32_t n_occ;          /* occupied orbitals of the WHOLE system, 0 < n_occ < N                                 */
    int32_t max_products;   /* 1 .. BML_SP2_LOG_LEN                                                                 */
    int32_t n_parts;        /* 1 .. BML_GRAPH_MAX_PARTS                                                             */
    int32_t part_capacity;  /* largest core+halo size the workspace is provisioned for (<= N)                       */
} bml_graph_sp2_params_t;

typedef struct {
    bml_sp2_stats_t sp2;    /* the shared SP2 record: status, products, branch bits, traces (over core orbitals), e_m */
    int32_t status;         /* = return value                                                                       */
    int32_t n_parts;
    int32_t overflow_row;   /* status -3: lowest row of D needing more than D->M slots, else -1                     */
    int32_t max_part_size;
    int32_t part_size[BML_GRAPH_MAX_PARTS];
    int32_t core_size[BML_GRAPH_MAX_PARTS];
} bml_graph_sp2_stats_t;

BML_API size_t bml_graph_sp2_workspace_bytes(int64_t N, int32_t n_parts, int32_t part_capacity);
BML_API int bml_graph_sp2_ellpack(const bml_matrix_t *H, const int32_t *d_core_offsets, const int32_t *d_core_nodes,
                                  const bml_graph_sp2_params_t *p, bml_matrix_t *D, void *d_workspace,
                                  size_t workspace_bytes, bml_graph_sp2_stats_t *stats, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* BML_GRAPH_H */
