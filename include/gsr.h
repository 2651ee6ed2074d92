/*
 * gsr.h -- C ABI of libgsr.so: the LSQR hot path of the Gaia AVU-GSR solver
 * (arXiv 2308.00778; citations are lines of /root/reference/PAPER.md) on one
 * NVIDIA B200 (sm_100a), FP64.
 *
 * The system  A x = b  (Eq. 1-3).  A has n_obs observation rows
 * and, below them, n_con constraint rows.  Every observation
 * row stores N_par = 24 coefficients in the section order
 *     [ 5 astrometric | 12 attitude = 3 axes x 4 | 6 instrumental | 1 global ]
 * and the unknowns are ordered
 *     [ astro: 5*n_stars | att axis0: n_dof_att | axis1 | axis2 | instr: n_instr | gamma ]
 * so n = 5*n_stars + 3*n_dof_att + n_instr + 1.  Coefficient k of row i is in column
 *     k <  5 : matrixIndexAstro[i] + k
 *     k < 17 : 5*n_stars + a*n_dof_att + matrixIndexAtt[i] + j,  a=(k-5)/4, j=(k-5)%4
 *     k < 23 : 5*n_stars + 3*n_dof_att + instrCol[6*i + (k-17)]
 *     k = 23 : 5*n_stars + 3*n_dof_att + n_instr
 * (index expressions of Algorithm 2).
 *
 * Model variants ("0 <= N_Astro <= 5", "0 <= N_Instr <= 6", N_Glob = 1 "or ... without
 * computing a global part"; runs with 5 global parameters; datasets that
 * solve only some of the sections).  gsr_layout carries the four section widths
 *     n_astro_par 0..5 | n_att_par 12 or 0 | n_instr_par 0..6 | n_glob_par 0..GSR_MAX_GLOB
 * and a row then stores N_par = their sum coefficients in the same section order.  A section of
 * width 0 has no columns: with kA = n_astro_par, kT = kA + n_att_par, kI = kT + n_instr_par,
 *     offAtt = n_astro_par*n_stars, offInstr = offAtt + (n_att_par ? 3*n_dof_att : 0),
 *     offGlob = offInstr + (n_instr_par ? n_instr : 0), n = offGlob + n_glob_par,
 *     k < kA : matrixIndexAstro[i] + k          (matrixIndexAstro[i] = n_astro_par*star(i))
 *     k < kT : offAtt + a*n_dof_att + matrixIndexAtt[i] + j,  a=(k-kA)/4, j=(k-kA)%4
 *     k < kI : offInstr + instrCol[n_instr_par*i + (k-kT)]
 *     else   : offGlob + (k-kI)                 (Alg. 2 "glob")
 * The production layout 5/12/6/1, 5/12/6/N_Glob for any other N_Glob, and the section subset
 * 0/12/6/0 run the specialised kernels (fused iteration, attitude copy); every other layout
 * runs one general pair of aprod kernels and the two-product iteration (its attitude section
 * still on the attitude copy; astrometric-only layouts have an aprod2 kernel of their own).
 *
 * Conventions
 *  - every call returns a gsr_status (0 = OK, negative = error); nothing throws;
 *    gsr_last_error(h) gives a handle-owned, NUL-terminated description.
 *  - "host or device" pointers are classified with cudaPointerGetAttributes;
 *    "device" pointers must be device memory of the handle's device.
 *  - the caller keeps ownership of every array it passes; the library copies.
 *  - a handle is not thread-safe; all work is ordered on the handle's stream and
 *    every call synchronises that stream before it returns.
 *  - there is no CPU fallback: without a CUDA device gsr_create fails (GSR_ECUDA).
 */
#ifndef GSR_H
#define GSR_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GSR_N_ASTRO 5
#define GSR_N_ATT 12
#define GSR_N_INSTR 6
#define GSR_N_GLOB 1
#define GSR_N_PAR 24
#define GSR_MAX_GLOB 16 /* widest global section a layout may ask for */

typedef enum {
    GSR_OK = 0,
    GSR_EINVAL = -1, /* bad argument (NULL, negative size, unsupported section width) */
    GSR_EINDEX = -2, /* an index array violates its contract; see gsr_bad_row()        */
    GSR_ENOMEM = -3, /* device or host allocation failed                               */
    GSR_ECUDA = -4,  /* CUDA runtime error (text in gsr_last_error)                    */
    GSR_ESTATE = -5  /* call order: e.g. aprod before upload, precondition twice       */
} gsr_status;

/* Sizes of one system.  Section widths: 5/12/6/1 is the production
 * layout (BASELINE north_star); see "Model variants" above for the others.  Widths outside
 * their ranges are GSR_EINVAL. */
typedef struct {
    int64_t n_obs;      /* observation rows m (>= 0)                                   */
    int64_t n_stars;    /* N_Stars (>= 1 when n_astro_par > 0)                         */
    int64_t n_dof_att;  /* N_DFA, attitude degrees of freedom per axis (>= 4 when
                           n_att_par > 0)                                              */
    int64_t n_instr;    /* number of instrumental columns (>= n_instr_par)             */
    int64_t n_con;      /* constraint rows appended below the observations (>= 0)      */
    int64_t n_con_nnz;  /* non-zeros of the constraint rows                            */
    int32_t n_astro_par, n_att_par, n_instr_par, n_glob_par; /* 5, 12, 6, 1 in production;
                           0..5, 12 or 0, 0..6, 0..GSR_MAX_GLOB in general             */
    int32_t device;     /* CUDA device ordinal                                         */
    uint32_t flags;     /* bitwise OR of GSR_FLAG_* (0 = default path)                 */
    void *stream;       /* cudaStream_t of the CALLER (e.g. torch's current stream), or
                           NULL for the legacy default stream.  The library always runs
                           on a non-blocking stream of its own; on entry every call
                           waits (cudaStreamSynchronize) for the work queued on THIS
                           stream, and it synchronises its own stream before it
                           returns.  Arguments produced on any other stream must be
                           complete before the call.                                   */
} gsr_layout;

/* gsr_layout.flags: per-handle choice of the kernel path (all paths compute the same
 * products; the tests run each of them against the oracle). */
#define GSR_FLAG_NO_ATT_COPY 1u /* do not build the block-time-ordered attitude copy
                                   (+104 B/row of HBM): aprod2 scatters the attitude
                                   section with atomics and gsr_lsqr runs the
                                   two-product iteration (low-memory path)            */
#define GSR_FLAG_NO_FUSE 2u     /* gsr_lsqr runs the two-product iteration (aprod1,
                                   then aprod2, as Alg. 1 l.17-25) instead of the
                                   fused single pass over A                            */
#define GSR_FLAG_INS_COPY 8u    /* build a column-ordered copy of the instrumental section
                                   (+72 B/row of HBM) and sum that section of A^T y on it
                                   without atomics (k_ins_scatter): bit-reproducible, but
                                   measured SLOWER than the default shared-memory / global
                                   atomics (Medium: 23.6 vs 21.3 ms per iteration), hence
                                   opt-in.  Needs the attitude copy, n_instr <= 65536 and
                                   unskewed columns; silently not built otherwise           */
#define GSR_FLAG_NO_TEX 4u      /* fused pass: gather the unknowns with plain loads
                                   instead of texture fetches (the path taken anyway
                                   when n >= 2^27 texels)                              */

typedef struct gsr_handle gsr_handle;

/* Outputs of gsr_lsqr.  x and se: caller-allocated, n doubles each, host or
 * device; se may be NULL. */
typedef struct {
    double *x;      /* solution of the original system (x = p (.) z, Alg. 1 l.27)      */
    double *se;     /* standard errors ("variances"; Alg. 1 l.26-27)      */
    int32_t istop;  /* Paige-Saunders stop code 0..7                                   */
    int64_t itn;    /* iterations done                                                 */
    double anorm, acond, rnorm, arnorm, xnorm; /* LSQR estimates (of the scaled system) */
} gsr_result;

/* Allocates the handle and all device storage for a system of these sizes.
 * PAPER.md:94-104 (Alg. 1 l.4-12: device selection, cudaMalloc). */
int32_t gsr_create(const gsr_layout *layout, gsr_handle **out);

/* Frees everything.  NULL is allowed. */
int32_t gsr_destroy(gsr_handle *h);

const char *gsr_last_error(const gsr_handle *h);

/* After GSR_EINDEX: first offending observation row (or -1). */
int64_t gsr_bad_row(const gsr_handle *h);

/* n (5*n_stars + 3*n_dof_att + n_instr + 1 in production; see "Model variants") and
 * m_tot = n_obs + n_con. */
int64_t gsr_ncols(const gsr_handle *h);
int64_t gsr_nrows(const gsr_handle *h);

/* Copies the system to the device (A_d, M_i, I_c; Alg. 1 l.6-12).
 *   values           f64 [n_obs*N_par] row-major, section order as above (N_par = the layout's
 *                    section widths summed; 24 in production)
 *   matrixIndexAstro i64 [n_obs]   = n_astro_par*star(i), non-decreasing (5*star(i) in production)
 *   matrixIndexAtt   i64 [n_obs]   = s_i in [0, n_dof_att-4] (axis-0 relative)
 *   instrCol         i32 [n_obs*n_instr_par] in [0, n_instr)
 *   b                f64 [n_obs+n_con] known terms
 * The index array of a section of width 0 is ignored and may be NULL.
 * All host or device.  Validates the index contracts on the device (GSR_EINDEX,
 * gsr_bad_row) and derives the star row pointer.  Replaces any earlier upload,
 * clears the preconditioned state and DISCARDS the constraint rows (gsr_precondition
 * scales them in place): call gsr_upload_constraints again after every upload. */
int32_t gsr_upload(gsr_handle *h, const double *values, const int64_t *matrixIndexAstro,
                   const int64_t *matrixIndexAtt, const int32_t *instrCol, const double *b);

/* Chunked form of gsr_upload for systems generated piecewise on the device (the
 * 116 GB "Large" config cannot exist twice in HBM): copies rows [row0, row0+nrows)
 * of the four arrays and of b.  Call gsr_upload_finish() once every row is in; it
 * validates and derives layouts exactly as gsr_upload does.  b_tail (n_con entries,
 * may be NULL when n_con == 0) holds the known terms of the constraint rows.
 * A new upload always starts from scratch: every row must come again before the next
 * gsr_upload_finish (the 4-byte star indices of the rows are upload scratch that the
 * finish step turns into the star row pointer and frees).  The ranges may come in any
 * order and may overlap (the last copy of a row counts); gsr_upload_finish returns
 * GSR_ESTATE, naming the first missing row, when some row has not been sent since the last
 * successful finish, and the handle stays unusable until the upload is completed.  After a
 * finish that failed with GSR_EINDEX the rows sent so far are kept: re-sending the offending
 * rows and calling gsr_upload_finish again is enough. */
int32_t gsr_upload_rows(gsr_handle *h, int64_t row0, int64_t nrows, const double *values,
                        const int64_t *matrixIndexAstro, const int64_t *matrixIndexAtt,
                        const int32_t *instrCol, const double *b);
int32_t gsr_upload_finish(gsr_handle *h, const double *b_tail);

/* Replaces the known terms b (n_obs+n_con doubles, host or device) of an uploaded system. */
int32_t gsr_set_b(gsr_handle *h, const double *b);

/* Constraint rows as CSR with absolute column indices:
 * rowptr i64 [n_con+1], col i64 [n_con_nnz] in [0, n), val f64 [n_con_nnz].
 * Host or device.  Must precede gsr_precondition. */
int32_t gsr_upload_constraints(gsr_handle *h, const int64_t *rowptr, const int64_t *col,
                               const double *val);

/* Derived layout, for bit-exact checks: i64 [n_stars+1], first row of each star.
 * out: host or device.  GSR_ESTATE when the layout has no astrometric section. */
int32_t gsr_get_star_rowptr(gsr_handle *h, int64_t *out);

/* Column preconditioning (Alg. 1 l.2-3): p_j = 1/||A_:j||_2 over all
 * rows including constraints (1 for an empty column), A_ij <- fl(A_ij * p_j) in
 * place on the device.  A second call is GSR_ESTATE. */
int32_t gsr_precondition(gsr_handle *h);

/* p (n doubles; all 1 before gsr_precondition).  out: host or device. */
int32_t gsr_get_colscale(gsr_handle *h, double *out);

/* Device copy of the matrix values as they stand (scaled if preconditioned):
 * out f64 [n_obs*N_par], host or device; con_val_out f64 [n_con_nnz] or NULL. */
int32_t gsr_get_values(gsr_handle *h, double *out, double *con_val_out);

/* aprod mode 1, Eq. 2, Algorithm 2:  y += A x  on the matrix as it
 * stands on the device.  x: n doubles, y: n_obs+n_con doubles, both DEVICE. */
int32_t gsr_aprod1(gsr_handle *h, const double *x, double *y);

/* aprod mode 2, Eq. 3, Algorithm 3:  x += A^T y.  DEVICE pointers.
 * The astrometric and global sections are summed in a fixed order (bit
 * reproducible); attitude and instrumental sums use floating-point atomics and
 * may differ in the last bits from run to run. */
int32_t gsr_aprod2(gsr_handle *h, const double *y, double *x);

/* LSQR of Paige & Saunders (Alg. 1 l.13-27) with damp = 0
 * on the device matrix and the uploaded b; b is not modified.  Runs at most itnlim
 * iterations; conlim <= 0 disables the condition-number test.  The whole iteration
 * (both aprods, norms, rotations, vector updates, stop tests) runs on the device;
 * the host only polls istop.  Writes x = p (.) z and se = p (.) se_z.
 * When the handle holds the block-time-ordered attitude copy, each iteration streams A's
 * row layout once: A^T u' is accumulated unscaled in the
 * pass that finishes u' = A v - alpha u, and 1/beta is applied to the n-vector afterwards
 * (same arithmetic up to rounding order; GSR_FLAG_NO_FUSE in gsr_layout.flags selects
 * the two-product form gsr_aprod1 / gsr_aprod2 expose). */
int32_t gsr_lsqr(gsr_handle *h, int64_t itnlim, double atol, double btol, double conlim,
                 gsr_result *result);

/* Covariances between couples of unknowns ("the covariances between the different couples of
 * unknowns are calculated"; Alg. 1 l.26-27).  The paper names neither the couples nor a formula:
 * the couples are the caller's, and the estimate is the one LSQR's variances are the diagonal of (Paige & Saunders'
 * sum_k d_k d_k^T, d_k = w_k / rho_k, which tends to (A'^T A')^-1), scaled like the standard errors:
 *     cov(i, j) = p_i p_j * rnorm^2 / (m_tot - n) * sum_k d_k[i] d_k[j]     (rnorm^2 alone when m_tot <= n),
 * so that cov(i, i) = se_i^2 (reading R26).
 * gsr_set_cov_pairs: npairs couples (pi[q], pj[q]) of column indices in [0, n), i64, host or device; the library
 * copies them.  They stay set for every later gsr_lsqr on this handle until replaced; npairs = 0 clears them.
 * GSR_EINDEX (gsr_last_error names the couple) for an index out of range.  Each iteration then costs one extra
 * kernel of npairs threads.  gsr_get_cov: the npairs covariances of the last gsr_lsqr, f64, host or device;
 * GSR_ESTATE before a solve with couples set. */
int32_t gsr_set_cov_pairs(gsr_handle *h, int64_t npairs, const int64_t *pi, const int64_t *pj);
int32_t gsr_get_cov(gsr_handle *h, double *out);

/* Per-iteration log of the last gsr_lsqr: up to max_itn rows of 5 doubles
 * (rnorm, arnorm, anorm, acond, xnorm) to a HOST buffer; returns rows written in
 * *n_written.  Only the last GSR_TRACE_CAP iterations are kept. */
#define GSR_TRACE_CAP 4096
int32_t gsr_get_trace(gsr_handle *h, double *out, int64_t max_itn, int64_t *n_written);

/* Which kernel path this handle uses (after gsr_upload): bit 0 = block-time-ordered
 * attitude copy in use, bit 1 = fused single-pass iteration, bit 2 = warp-level
 * pre-summation of equal instrument columns (chosen from the column histogram at
 * upload), bit 3 = texture gathers in the fused pass, bit 4 = 2-byte instrument
 * columns on the device, bit 5 = the fused iteration keeps a copy of u in block-time
 * order for the attitude kernel (+8 B/row of HBM; dropped when it does not fit). */
#define GSR_PATH_ATT_COPY 1
#define GSR_PATH_FUSED 2
#define GSR_PATH_INSTR_MATCH 4
#define GSR_PATH_TEX 8
#define GSR_PATH_IC16 16
#define GSR_PATH_UT 32
#define GSR_PATH_INS_COPY 64 /* column-ordered copy of the instrumental section in use
                                (GSR_FLAG_INS_COPY): that section of A^T y is summed without
                                atomics and is bit-reproducible                               */
int32_t gsr_path_info(const gsr_handle *h);

/* Device time of the last gsr_lsqr's iteration loop in milliseconds (CUDA events on
 * the handle's stream), and the number of kernels launched in it. */
int32_t gsr_last_timing(gsr_handle *h, double *loop_ms, int64_t *kernel_launches);

#ifdef __cplusplus
}
#endif
#endif /* GSR_H */
