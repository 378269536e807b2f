/*
 * qmc_b200.h -- C ABI of libqmcb200.so: the data-parallel hot path of the real-space
 * VMC/DMC particle-by-particle move (arxiv 1802.06922, "QMCPACK: an open source ab initio
 * quantum Monte Carlo package ..."), hand-written CUDA for one B200 (sm_100a).
 *
 * Citations are PAPER.md line numbers (+ section / equation).  "R:Ax" is a reading listed in
 * DESIGN.md section 3, used where the paper is silent.
 *
 * Conventions for every call
 *   - returns QMC_OK (0) or a negative QMC_E* code; qmc_last_error() gives a thread-local
 *     message.  Never aborts, never throws, never falls back to the CPU.
 *   - "dev" pointers are CUDA device pointers on the current device, "host" pointers are
 *     ordinary host memory.  Every buffer passed in is caller-owned; handles own their
 *     internal device storage until the matching *_destroy call.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls
 *     enqueue work on it and do not synchronise unless stated.
 *   - all arrays are dense row-major with the stated leading dimensions.
 *   - one GPU; walkers are independent Markov chains (L181), so multi-GPU use is one library
 *     instance per rank with the walkers partitioned.
 */
#ifndef QMC_B200_H
#define QMC_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QMC_OK 0
#define QMC_EINVAL (-1)    /* bad argument (shape, alignment, NULL, handle mismatch)      */
#define QMC_ENOMEM (-2)    /* device or host allocation failed                            */
#define QMC_ECUDA (-3)     /* a CUDA runtime call failed; message holds cudaGetErrorString */
#define QMC_ESINGULAR (-4) /* a Slater matrix had a zero / non-finite pivot in qmc_det_init */

#define QMC_MAX_DELAY 32   /* largest delayed-update rank accepted by qmc_det_init        */

typedef struct qmc_spline qmc_spline_t; /* opaque: padded fp32 coefficient table on device */
typedef struct qmc_det qmc_det_t;       /* opaque: per-walker fp64 inverse + scratch       */
typedef struct qmc_jastrow qmc_jastrow_t; /* opaque: Jastrow function table + ions on device */

/* Thread-local text of the last error raised on this thread ("" if none). */
const char *qmc_last_error(void);

/* ---------------------------------------------------------------------------------------
 * qmc_spline_create -- PAPER.md L307-311 (sec 6.2.1): single-particle orbitals "converted into
 * a regular 3D B-spline representation in real-space"; "spline coefficients may also be stored
 * in single precision" (L311); one read-only table per GPU shared by all walkers (L311, L114).
 *
 *   nx,ny,nz   grid points per cell edge (>= 1; periodic, L307)
 *   norb       number of orbitals N (>= 1)
 *   lattice    host, 9 doubles row-major, rows = cell vectors a0,a1,a2 (r = u . lattice);
 *              must be invertible.  General (skewed) cells are supported (R:A5).
 *   coefs      canonical table float [nx][ny][nz][norb], orbital index innermost, periodic,
 *              no halo (R:A3, R:A4); host memory if coefs_on_device == 0, else device memory.
 *   The library builds and OWNS a padded device copy [nx][ny][nz][Np], Np = norb rounded up
 *   to a multiple of 32 floats (128-byte rows; pad = 0), so the caller may free `coefs` after
 *   the stream has drained.  With coefs_on_device != 0 and norb % 32 == 0 the padded copy is a
 *   plain device-to-device copy.
 * Errors: QMC_EINVAL (sizes, NULL, singular lattice), QMC_ENOMEM, QMC_ECUDA.
 */
int qmc_spline_create(qmc_spline_t **out, int nx, int ny, int nz, int norb,
                      const double *lattice, const float *coefs, int coefs_on_device,
                      void *stream);
int qmc_spline_destroy(qmc_spline_t *spline);
/* qmc_spline_set_half_twist -- PAPER.md L449-455 (sec 9.2, eq. 43): real orbitals at a half twist,
 * twist angle Theta_d = K . a_d = pi along every cell vector d with half_twist[d] == 1 and 0 along
 * the others, so phi(r + a_d) = -phi(r) there (reading R:A23 in DESIGN.md).  The table then holds one
 * cell of an antiperiodic function: control points reached across the face of cell vector d, and
 * positions in odd images of the cell, take the factor -1 in every later evaluation through this
 * handle (qmc_spo_vgl, qmc_det_*, qmc_sweep*): ratios, inverses and sweeps follow unchanged.
 *   half_twist   host, 3 ints, each 0 or 1; {0,0,0} (the state after qmc_spline_create) is periodic.
 * Host-side flag only: no device work, no allocation; set it before the first launch that uses the
 * handle, not while one is in flight.  General twists need complex orbitals: DESIGN.md section 9.
 * Errors: QMC_EINVAL (NULL, a value other than 0 / 1).
 */
int qmc_spline_set_half_twist(qmc_spline_t *spline, const int *half_twist);
/* Row pitch Np (floats) and bytes of the padded device table; either pointer may be NULL. */
int qmc_spline_info(const qmc_spline_t *spline, int *row_pitch, size_t *table_bytes);

/* ---------------------------------------------------------------------------------------
 * qmc_spo_vgl -- value, Cartesian gradient and Laplacian of all N orbitals at npos positions:
 * "a constant 64 coefficients to be accessed in memory to evaluate each single-particle
 * wavefunction" (L309).  Uniform cubic B-spline (R:A1), control points i..i+3 (mod N_d) per
 * dimension with i = floor(s), s = frac(r . lattice^-1) * N_d (R:A2, the support convention of
 * eq. 33; R:A7 at cell faces).  Index and fraction in fp64, the 64 x {v,gx,gy,gz,lap}
 * stencil weights rounded to fp32, fp32 accumulation in a fixed order (bit-reproducible,
 * independent of the batch, R:A11).
 *
 *   pos   dev, double [npos][3], Cartesian, any image of the cell
 *   v     dev, float [npos][ldo]        phi_n(r_p)
 *   g     dev, float [npos][3][ldo]     d phi_n / d r_j ; may be NULL
 *   l     dev, float [npos][ldo]        Laplacian        ; may be NULL (g and l together)
 *   ldo   leading dimension of the outputs: >= norb, multiple of 4; v,g,l 16-byte aligned.
 *         Elements norb..ldo-1 of each row are written with zeros up to the table pitch.
 * npos == 0 is a no-op.  Errors: QMC_EINVAL, QMC_ECUDA.
 */
int qmc_spo_vgl(const qmc_spline_t *spline, int npos, const double *pos, float *v, float *g,
                float *l, int ldo, void *stream);

/* ---------------------------------------------------------------------------------------
 * qmc_det_init -- Slater matrices M_ij = phi_j(r_i) (L325) of nwalkers walkers ("multiple
 * walkers can be assigned to each GPU", L114), their inverses in fp64, log|det| and sign.
 *
 *   nel         electrons in this determinant; must equal the spline's norb
 *   pos         dev, double [nwalkers][nel][3]
 *   delay_rank  0 or 1: Sherman-Morrison rank-1 update on every accepted move (L299, [49]);
 *               2..QMC_MAX_DELAY: delayed update (L112, L299, [44]) -- accepted rows are
 *               buffered and applied as one rank-k contraction (R:A14).
 * The handle owns B_w = (A_w^-1)^T as double [nwalkers][nel][ld] (row k of B is column k of
 * A^-1, "the moved electron's inverse-matrix row"), ld = nel rounded up to 64 doubles, pad 0.
 * The orbital values come from qmc_spo_vgl (fp32, upcast; R:A16); the inverse is an in-place
 * Gauss-Jordan elimination with partial pivoting, all on the device.
 * Synchronises `stream` once (to report singularity).
 * Errors: QMC_EINVAL, QMC_ENOMEM, QMC_ECUDA, QMC_ESINGULAR (handle not created).
 */
int qmc_det_init(qmc_det_t **out, const qmc_spline_t *spline, int nwalkers, int nel,
                 const double *pos, int delay_rank, void *stream);
int qmc_det_destroy(qmc_det_t *det);

/* ---------------------------------------------------------------------------------------
 * qmc_det_init_ex -- qmc_det_init with flags.  QMC_DET_FP32_INVERSE: "the numerical
 * precision is parameterized, with single, double and mixed precision": the handle STORES
 * B = (A^-1)^T in fp32, float [nwalkers][nel][ld] (half the bytes every update and flush moves; reading
 * R:A19 of DESIGN.md): the initial inverse is computed in fp64 and rounded once; every kernel converts
 * the rows it reads to fp64, does all arithmetic (ratios, Sherman-Morrison multipliers, the tensor-core
 * contractions of the delayed update, log|det|) in fp64, and rounds to nearest even when it stores --
 * after every accepted update (delay_rank <= 1) or once per window flush (delay_rank >= 2).  The
 * rounding error accumulates slowly: monitor it with qmc_det_residual and refresh the inverse from the
 * positions with qmc_det_recompute every few sweeps.
 */
#define QMC_DET_FP32_INVERSE 1u
/* QMC_DET_ACCEPT_WINDOWS (with 2 <= delay_rank <= 16; reading R:A14 of DESIGN.md): a window of the delayed update
 * closes when the walker has ACCEPTED delay_rank moves (or after 3/2 delay_rank steps, or at the end of the
 * sweep) instead of after delay_rank steps, so that every flush applies a full window: the one pass over the
 * inverse is amortised over delay_rank accepted moves, not over 0.8 delay_rank.  The walkers of a handle then
 * advance through the electrons at their own pace (a per-walker cursor on the device; the SPO-VGL scratch is a
 * ring indexed by electron, so every proposal is still evaluated once); decisions, ratios and the inverse are
 * the same as with any other window choice.  qmc_sweep* only. */
#define QMC_DET_ACCEPT_WINDOWS 2u
int qmc_det_init_ex(qmc_det_t **out, const qmc_spline_t *spline, int nwalkers, int nel,
                    const double *pos, int delay_rank, unsigned flags, void *stream);
/* 8 (fp64 inverse) or 4 (QMC_DET_FP32_INVERSE). */
int qmc_det_storage(const qmc_det_t *det, int *bytes_per_element);

/* qmc_det_recompute -- the inverse, log|det| and sign of every walker again from scratch at `pos`
 * (dev, double [nwalkers][nel][3]), exactly as qmc_det_init computes them (Slater matrix from the SPO
 * kernel, Gauss-Jordan in fp64, rounded once for fp32 storage); the accept counters are kept and an
 * open delayed window is closed first.  The "recompute" of mixed precision (L82; R:A19) and of
 * north_star's residual check.  Synchronises `stream`.  QMC_ESINGULAR leaves the inverse undefined. */
int qmc_det_recompute(qmc_det_t *det, const qmc_spline_t *spline, const double *pos, void *stream);

/* qmc_det_residual -- drift monitor: resid_out[w] (dev, double [nwalkers]) =
 *     max over the nsample electrons i = s * (nel / nsample) and all k of | B_w[k] . phi(r_i) - delta_ik |
 * i.e. nsample rows of A B^T - I with A recomputed by the SPO kernel at `pos` (R:A11); one pass over B
 * per call.  nsample * nel * 8 bytes must fit 96 KB of shared memory.  Pending delayed updates are
 * applied first.  Synchronises `stream`. */
int qmc_det_residual(qmc_det_t *det, const qmc_spline_t *spline, const double *pos, int nsample,
                     double *resid_out, void *stream);

/* ---------------------------------------------------------------------------------------
 * qmc_det_ratio -- L299: for a single-electron move of electron iel to a position where the
 * orbitals take the values phi, det A'/det A = sum_j B[iel][j] * phi[j] (fp64 accumulation of
 * the upcast fp32 orbital vector; warp-shuffle tree, fixed order).  With a delayed window open
 * the pending accepted rows are included (R:O7).
 *
 *   phi    dev, float [nwalkers][ldo], ldo >= nel.  With delay_rank >= 2 (here and in
 *          qmc_det_accept_update) the vector is read with 128-bit loads up to the table pitch and
 *          copied into the window: ldo >= the spline's row pitch (qmc_spline_info), ldo % 4 == 0,
 *          phi 16-byte aligned, elements nel..pitch-1 finite (qmc_spo_vgl writes zeros there);
 *          otherwise QMC_EINVAL.
 *   ratio  dev, double [nwalkers] (out)
 */
int qmc_det_ratio(qmc_det_t *det, int iel, const float *phi, int ldo, double *ratio,
                  void *stream);

/* ---------------------------------------------------------------------------------------
 * qmc_det_ratio_points -- ratio-only evaluation of several trial positions of ONE electron against
 * the same inverse row, with no update: the access pattern of the semi-local pseudopotential
 * quadrature ("a 12 point angular integration used by default"), where every
 * quadrature point needs det A'/det A = sum_j B[iel][j] * phi_q[j] (L299) and nothing else.
 * Evaluate the orbital values of the nwalkers * npts points with qmc_spo_vgl (g = l = NULL) first.
 *
 *   phi     dev, float [nwalkers][npts][ldo], ldo >= nel
 *   ratios  dev, double [nwalkers][npts] (out)
 * With delay_rank >= 2 the pending accepted rows are applied first (the inverse is made current).
 */
int qmc_det_ratio_points(qmc_det_t *det, int iel, int npts, const float *phi, int ldo,
                         double *ratios, void *stream);

/* ---------------------------------------------------------------------------------------
 * qmc_det_accept_update -- L299 "for single electron moves, QMCPACK uses the Sherman-Morrison
 * algorithm": for every walker with accept[w] != 0, row iel of A_w is replaced by phi_w and
 *     B'[m][j] = B[m][j] - ((B[m] . phi) - delta_{m,iel}) * B[iel][j] / ratio_w
 * in ONE pass over B (each row read once, dotted, updated, written: 16*nel*ld bytes per
 * accepted walker).  log|det| += log|ratio|, sign *= sgn(ratio), accept counter += 1.
 * Walkers with accept[w] == 0 are untouched, and so are walkers whose ratio is zero or not finite
 * (the update divides by it and the new Slater matrix would be singular: the accept is refused,
 * R:A18; the same holds for forced_accept in qmc_sweep).  With delay_rank >= 2 the row is appended
 * to the walker's window instead and the window is flushed when any walker's window is full.
 *
 *   phi, ldo  as in qmc_det_ratio (the vector the ratio was computed from)
 *   ratio     dev, double [nwalkers]: the values qmc_det_ratio returned
 *   accept    dev, unsigned char [nwalkers]
 */
int qmc_det_accept_update(qmc_det_t *det, int iel, const float *phi, int ldo,
                          const double *ratio, const unsigned char *accept, void *stream);

/* Apply all pending delayed updates (no-op for delay_rank <= 1). */
int qmc_det_flush(qmc_det_t *det, void *stream);

/* ---------------------------------------------------------------------------------------
 * qmc_sweep -- L195-199 (sec 5.2.1): "particle-by-particle moves work by iterating
 * sequentially over all electrons"; all walkers advance in lockstep (L114, L181).  For sweep s,
 * electron k, walker w:  r' = pos[w][k] + delta[s][k][w]  (eq. 13 with F = 0, pre-generated
 * Gaussian);  phi, grad, lap = SPO-VGL(r');  R = B_w[k] . phi;  accept iff R*R > u[s][k][w]
 * (eq. 12 with symmetric T and a determinant-only Psi, R:A8; non-finite R rejects); on accept
 * pos[w][k] = r' (stored unwrapped) and the inverse is updated as in qmc_det_accept_update.
 * Pending delayed updates are flushed at the end of every sweep.  qmc_sweep_ex adds the fixed-node
 * rule (L253) and the wavefunction force of every proposal (L156) as options.
 *
 *   pos            dev, double [nwalkers][nel][3], in/out.  Must be the positions the handle's
 *                  inverse corresponds to.
 *   delta          dev, double [nsweeps][nel][nwalkers][3]
 *   uniforms       dev, double [nsweeps][nel][nwalkers], in [0,1)
 *   ratios_out     dev, double [nsweeps][nel][nwalkers] or NULL
 *   accept_out     dev, unsigned char, same shape, or NULL
 *   forced_accept  NULL, or dev unsigned char (same shape): decisions to impose instead of the
 *                  Metropolis test (parity protocol)
 */
int qmc_sweep(qmc_det_t *det, const qmc_spline_t *spline, double *pos, const double *delta,
              const double *uniforms, int nsweeps, double *ratios_out,
              unsigned char *accept_out, const unsigned char *forced_accept, void *stream);

/* Options of qmc_sweep_ex; zero-initialise for the qmc_sweep behaviour. */
typedef struct qmc_sweep_opts {
    int iel_begin;       /* first electron moved in each sweep (default 0)                   */
    int iel_count;       /* electrons moved per sweep; 0 = nel - iel_begin                   */
    float *phi_record;   /* NULL, or dev float [nsweeps][nel][nrecord][nel]: the fp32 orbital */
    int nrecord;         /*   vector of every move of walkers 0..nrecord-1 (parity replay)   */
    int fixed_node;      /* != 0: fixed-node rule: a move that changes the   */
                         /*   sign of the wavefunction (R < 0) is rejected whatever u is     */
    double *force_out;   /* NULL, or dev double [nsweeps][nel][nwalkers][3]: the wavefunction */
                         /*   force F = 2 grad log Psi_T (L156; the F of eq. 11 / eq. 13) on  */
                         /*   the moved electron at the PROPOSED configuration,               */
                         /*   F = 2 sum_j grad phi_j(r') B[k][j] / R, for every move          */
                         /*   (accepted or not; 0 where R == 0)                               */
    double drift_tau;    /* > 0: drift moves (reading R:A20).  `delta` then holds   */
                         /*   the diffusion part chi ~ N(0, tau) per component and the proposal is      */
                         /*   r' = r_k + tau F_k(r) + chi  (eq. 13 / eq. 19 with lambda = 1/2), with     */
                         /*   F_k(r) = 2 grad_k log Psi_T = 2 sum_j grad phi_j(r_k) B[k][j] (L156) at    */
                         /*   the CURRENT configuration; the move is accepted iff (eq. 12)              */
                         /*   R^2 T(r'->r)/T(r->r') > u,  log T'/T = (|r' - r - tau F(r)|^2              */
                         /*   - |r - r' - tau F(r')|^2) / (2 tau).  One SPO-VGL gather more per move    */
                         /*   (gradients at the current position, batched over 16 electrons) and the     */
                         /*   proposal gather per step (it depends on the decisions before it).          */
                         /*   With delay_rank >= 2 pending rows are applied first and every step is a   */
                         /*   rank-1 update (the one-launch window needs all its proposals up front).    */
    double *rprop_out;   /* NULL, or dev double [nsweeps][nel][nw][3]: the proposed positions (drift)   */
    double *logt_out;    /* NULL, or dev double [nsweeps][nel][nw]: log T(r'->r)/T(r->r') (drift)       */
    double *fcur_out;    /* NULL, or dev double [nsweeps][nel][nw][3]: F_k(r) at the current config.    */
    const struct qmc_jastrow *jastrow;   /* NULL, or a Jastrow factor (qmc_jastrow_create): Psi_T = e^{-J} D      */
                         /*   (eq. 26, eq. 28-33), so |Psi'/Psi|^2 = R^2 exp(-2 dJ) and the move is     */
                         /*   accepted iff R^2 exp(-2 dJ) > u (eq. 12, symmetric T), dJ taken at the walker's    */
                         /*   CURRENT configuration.  ratios_out stays the determinant ratio R.  Rank-1 mode: one */
                         /*   more small launch per step; delayed mode: one launch per window (dJ of its K        */
                         /*   proposals against the window-start configuration) and an O(p) correction per step   */
                         /*   inside the window kernel for the electrons the window has already moved.  Not with  */
                         /*   drift_tau > 0 (the drift would need grad J): QMC_EINVAL.                            */
    const double *jastrow_other;   /* NULL, or dev double [nw][jastrow_nother][3]: the electrons of the other    */
    int jastrow_nother;            /*   spin (fixed during this sweep; opposite-spin function).  qmc_wf_sweep    */
                                   /*   fills both in from the other determinant's positions.                    */
    double *jratio_out;  /* NULL, or dev double [nsweeps][nel][nw]: exp(-dJ) of every move                        */
} qmc_sweep_opts_t;

int qmc_sweep_ex(qmc_det_t *det, const qmc_spline_t *spline, double *pos, const double *delta,
                 const double *uniforms, int nsweeps, double *ratios_out,
                 unsigned char *accept_out, const unsigned char *forced_accept,
                 const qmc_sweep_opts_t *opts, void *stream);

/* Same as qmc_sweep with HOST buffers (pos in/out; ratios_out / accept_out may be NULL):
 * copies the inputs to the device, runs the sweeps, copies pos, ratios and decisions back and
 * synchronises `stream`.  Host buffers should be page-locked for full copy bandwidth. */
int qmc_sweep_host(qmc_det_t *det, const qmc_spline_t *spline, double *pos_host,
                   const double *delta_host, const double *uniforms_host, int nsweeps,
                   double *ratios_out_host, unsigned char *accept_out_host, void *stream);

/* ---------------------------------------------------------------------------------------
 * State access (checkpoint / parity).  Pending delayed updates are flushed first.
 *   qmc_det_get_inverse   binv_out dev double [nwalkers][nel][nel] dense, B = (A^-1)^T (fp32 storage:
 *                         upcast exactly; set_inverse rounds to nearest even)
 *   qmc_det_set_inverse   the reverse (binv_in dense); logdet / sign dev arrays or NULL (kept)
 *   qmc_det_get_stats     dev: logdet double [nwalkers], sign int [nwalkers],
 *                         naccept long long [nwalkers]; any may be NULL
 *   qmc_det_info          nwalkers, nel, ld (doubles), delay_rank; any may be NULL
 */
int qmc_det_get_inverse(qmc_det_t *det, double *binv_out, void *stream);
int qmc_det_set_inverse(qmc_det_t *det, const double *binv_in, const double *logdet,
                        const int *sign, void *stream);
int qmc_det_get_stats(qmc_det_t *det, double *logdet, int *sign, long long *naccept,
                      void *stream);
int qmc_det_info(const qmc_det_t *det, int *nwalkers, int *nel, int *ld, int *delay_rank);

/* ---------------------------------------------------------------------------------------
 * qmc_det_kinetic -- the determinant's kinetic term of the local energy, eq. 3 (first
 * term, -1/2 sum_i lap_i) and eq. 37 (E_L,n = Psi_T^-1 H_n Psi_T), "collected after all Monte Carlo
 * walkers have advanced one step" (L401).  For Psi = det A only row i of A depends on r_i:
 *     grad_out[w][i][:] = grad_i det A / det A = sum_j grad phi_j(r_i) B[i][j]
 *     lap_out[w][i]     = lap_i  det A / det A = sum_j lap  phi_j(r_i) B[i][j]
 *     one_out[w][i]     = sum_j phi_j(r_i) B[i][j]        (= 1 when B is the inverse at pos)
 *     ekin_out[w]       = -1/2 sum_i lap_out[w][i]         (Hartree; determinant-only Psi)
 * The SPO-VGL of the CURRENT positions is evaluated in fp32 by the sweep's batched gather kernel
 * and contracted in fp64 (fixed order).  Pending delayed updates are flushed first.
 *
 *   pos       dev, double [nwalkers][nel][3]: the positions the handle's inverse corresponds to
 *   grad_out  dev, double [nwalkers][nel][3] or NULL;   lap_out, one_out  dev, double [nwalkers][nel] or NULL
 *   ekin_out  dev, double [nwalkers] or NULL            (at least one output must be given)
 */
int qmc_det_kinetic(qmc_det_t *det, const qmc_spline_t *spline, const double *pos, double *grad_out,
                    double *lap_out, double *one_out, double *ekin_out, void *stream);

/* qmc_det_kinetic_noalloc -- ekin_out of qmc_det_kinetic (eq. 3 first term, eq. 37) for callers that may not
 * allocate device memory (code under CUDA graph capture, serving loops, harnesses that forbid it).
 * qmc_det_kinetic(..., lap_out = NULL, ...) takes its per-electron Laplacian scratch from cudaMalloc on the
 * handle's first such call; this entry point calls no cudaMalloc, cudaFree or allocating library routine:
 * the scratch is a file-scope device array of QMC_KINETIC_NOALLOC_MAX doubles (4 MiB) inside the library
 * image, which every GPU that loads the library holds until the process exits.  Same kernels and summation
 * order as qmc_det_kinetic: ekin_out has the same bits.
 *
 *   pos       dev, double [nwalkers][nel][3] (as qmc_det_kinetic);  ekin_out  dev, double [nwalkers] (caller's)
 *   The handle's device must be the current device.
 *   nwalkers * nel > QMC_KINETIC_NOALLOC_MAX: QMC_EINVAL, nothing launched (use qmc_det_kinetic).
 *   All calls on a device share the one array.  A call overwrites every element it reads, so nothing carries
 *   over from call to call, but calls that overlap on the GPU (different streams or host threads, also on
 *   different handles) race on it: keep them on one stream or order them with events.
 * Errors: QMC_EINVAL, QMC_ECUDA. */
#define QMC_KINETIC_NOALLOC_MAX (1 << 19) /* elements = nwalkers * nel; `large` (512 x 1024) just fits */
int qmc_det_kinetic_noalloc(qmc_det_t *det, const qmc_spline_t *spline, const double *pos, double *ekin_out,
                            void *stream);

/* ---------------------------------------------------------------------------------------
 * qmc_wf_* -- the product of two spin determinants, Psi_T = D_up D_dn: PAPER.md eq. 26 (L295),
 * Psi_T = sum_i c_i D_i^up D_i^dn e^J with one determinant per spin and no Jastrow factor.  A sweep
 * iterates "sequentially over all electrons" (L195): the nup electrons of the up determinant, then the
 * ndn of the down determinant; moving an up electron leaves D_dn unchanged, so the ratio of the move is
 * D_up'/D_up and only that inverse is updated.  The handle does NOT own the determinants or the splines
 * (each spin has its own orbital set; pass the same spline twice for a closed shell), which must have
 * the same walker count and live on the same device.
 *
 *   qmc_wf_sweep    pos_up dev double [nw][nup][3], pos_dn dev double [nw][ndn][3] (in/out);
 *                   delta dev double [nsweeps][nup+ndn][nw][3], uniforms / ratios_out / accept_out /
 *                   forced_accept [nsweeps][nup+ndn][nw] (electron index: up first); opts as in
 *                   qmc_sweep_ex (fixed_node, force_out, drift_tau and its outputs, jastrow and
 *                   jratio_out, with the [nup+ndn] electron axis; iel_begin / iel_count / phi_record
 *                   must be 0 / NULL; jastrow_other / jastrow_nother are filled in by the call: the
 *                   other determinant's electrons at their current positions).
 *   qmc_wf_kinetic  ekin_out dev double [nw] = -1/2 sum over ALL electrons of lap_i Psi / Psi (eq. 3),
 *                   the sum of the two determinants' qmc_det_kinetic.
 *   qmc_wf_get_stats  logpsi dev double [nw] = log|D_up| + log|D_dn|, sign dev int [nw] = their
 *                   product; either may be NULL.
 */
typedef struct qmc_wf qmc_wf_t;
int qmc_wf_create(qmc_wf_t **out, qmc_det_t *det_up, const qmc_spline_t *spline_up, qmc_det_t *det_dn,
                  const qmc_spline_t *spline_dn);
int qmc_wf_destroy(qmc_wf_t *wf);
int qmc_wf_info(const qmc_wf_t *wf, int *nwalkers, int *nup, int *ndn);
int qmc_wf_sweep(qmc_wf_t *wf, double *pos_up, double *pos_dn, const double *delta, const double *uniforms,
                 int nsweeps, double *ratios_out, unsigned char *accept_out,
                 const unsigned char *forced_accept, const qmc_sweep_opts_t *opts, void *stream);
int qmc_wf_kinetic(qmc_wf_t *wf, const double *pos_up, const double *pos_dn, double *ekin_out, void *stream);
int qmc_wf_get_stats(qmc_wf_t *wf, double *logpsi, int *sign, void *stream);

/* ---------------------------------------------------------------------------------------
 * qmc_jastrow_* -- one- and two-body Jastrow factor with cubic B-spline functors, sec 7:
 * Psi = e^{-J} Phi (eq. 28, eq. 29), J = sum_i u_1(r_i) + 1/2 sum_{i != j} u_2(r_i, r_j) (eq. 30 up to the
 * two-body term), u_1(r_i) = sum_I u_{species(I)}(|r_i - R_I|) (eq. 31), u_2 = u_{ss'}(|r_i - r_j|) (eq. 32,
 * first term; one function for equal spins and one for opposite spins, L365), each functor
 *     u(r) = sum_{m=0}^{M} p_m B_3(r / (r_c / M) - m),   B_3 the cardinal cubic B-spline on [-3, 1)   (eq. 33)
 * and u = 0 for r >= r_c (reading R:A21).  Periodic cells use the nearest image of every pair ("the cutoffs
 * must be smaller than the simulation cell Wigner-Seitz radius", L375); lattice == NULL is open boundaries.
 * The three-body term (eq. 32 second term, eq. 35) is not built.
 *
 *   qmc_jastrow_create  all arguments HOST: lattice 9 doubles (rows = cell vectors) or NULL; nfunc <= 8
 *                       functors with cutoffs rc[f], M[f] >= 1 intervals and control points
 *                       p[sum_{g<f}(M[g]+1) .. + M[f]] (at most 256 - 4 nfunc in all); f_same / f_opp: the
 *                       electron-electron functors (-1 = none); nion ions at ion_pos [nion][3] with functor
 *                       ion_func [nion] (-1 = none).  Copies everything to the current device.
 *   qmc_jastrow_ratio   the move of electron iel of every walker to rnew (dev double [nwalkers][3]):
 *                       dj_out[w] = J(R') - J(R) = the terms of eq. 30 that contain the electron, at rnew minus at
 *                       pos[w][iel]; ratio_out[w] = exp(-dJ) = the Jastrow part of Psi'/Psi.  pos dev double
 *                       [nwalkers][nel][3] (one spin); other dev double [nwalkers][nother][3] (the other spin)
 *                       or NULL with nother = 0.  Either output may be NULL.  One launch, fp64, fixed order.
 *   qmc_jastrow_value   j_out[w] = J of walker w (dev double [nwalkers]); O(N^2), for checks.
 * In a sweep: qmc_sweep_opts_t.jastrow (above).
 */
int qmc_jastrow_create(qmc_jastrow_t **out, const double *lattice, int nfunc, const double *rc, const int *M,
                       const double *p, int f_same, int f_opp, int nion, const double *ion_pos,
                       const int *ion_func);
int qmc_jastrow_destroy(qmc_jastrow_t *jastrow);
int qmc_jastrow_ratio(const qmc_jastrow_t *jastrow, int nwalkers, int nel, const double *pos, int nother,
                      const double *other, int iel, const double *rnew, double *ratio_out, double *dj_out,
                      void *stream);
int qmc_jastrow_value(const qmc_jastrow_t *jastrow, int nwalkers, int nel, const double *pos, int nother,
                      const double *other, double *j_out, void *stream);

/* ---------------------------------------------------------------------------------------
 * Per-kernel timing of qmc_sweep* (bench.py's roofline): with profiling enabled every kernel
 * launch of a sweep is bracketed by CUDA events on the launching stream.
 *   qmc_det_profile(det, 1)   enable and reset;  (det, 0) disable
 *   qmc_det_profile_read      synchronises the recorded events and returns, per kernel kind,
 *                             the summed device time in ms and the number of launches; host
 *                             arrays of QMC_PROF_KINDS entries.  Kinds: 0 SPO-VGL of a batch of
 *                             electron steps, 1 rank-1 update, 2 delayed ratio/decide/append,
 *                             3 delayed accept (standalone), 4 delayed flush, 5 ratio + row copy.
 *                             In qmc_sweep kind 2 is the one-launch-per-window kernel (ratios, decisions and
 *                             moves of K steps).
 *                             Resets the recorder.
 */
#define QMC_PROF_KINDS 6
int qmc_det_profile(qmc_det_t *det, int enable);
int qmc_det_profile_read(qmc_det_t *det, double *ms_host, long long *launches_host);

/* Environment variables read by qmc_det_flush / qmc_sweep (test and A/B-measurement hooks only; unset
 * in production): QMC_FLUSH_RING=0 routes every shape to the shared-memory-window flush kernel
 * (flush.cu) instead of the register-window / TMA-ring kernel (flush_ring.cu); QMC_FLUSH_SHAPE=n
 * forces the n-th launch shape of flush.cu for the handle's leading dimension; QMC_FLUSH_LAG=0 selects
 * the round-1 ring kernel (reduction by two compute warps), 1 / 2 the lag between the two contractions in
 * the warp-specialised ring kernel (default 1), QMC_FLUSH_PP=1 its ping-pong variant; QMC_FLUSH_HP=1
 * routes ranks 17..32 to the helper-pipelined kernel (flush_ring_hp.cu) instead of flush_ring_hi.cu;
 * QMC_SWEEP_OVERLAP=0 keeps the next window's SPO-VGL on the sweep's own stream.  Results are the same
 * to rounding with any setting (tests/test_gpu_parity.py::test_delayed_large_n_equals_rank1). */

/* Measured fp64 tensor-core peak of the current device in TFLOP/s (host pointer): an issue loop of
 * mma.sync.m8n8k4.f64 with register operands, best of 5 after a warm-up, ~10 ms.  bench.py reports
 * the delayed flush (the "genuine dense fp64 contraction" of north_star) against it,
 * since MEASURED_PEAKS.json holds no fp64 figure.  Synchronises the stream. */
int qmc_probe_fp64_dmma(double *tflops_host, void *stream);
/* The fp64 pipe of an SM sub-partition under different mixes (what the flush kernels are laid out around;
 * profiles/r02_fp64_pipe.md): mode 0 = DMMA.8x8x4 only, 1 = DFMA only, 2 = one DMMA + two DFMA per slot;
 * warps_per_sm in 1..32 (one CTA per SM), chains in {1, 2, 4, 8} independent accumulators per warp.  Returns
 * the DMMA and the DFMA throughput in TFLOP/s (host pointers; 0 for the absent instruction).  Synchronises. */
int qmc_probe_fp64_pipe(int mode, int warps_per_sm, int chains, double *tflops_dmma_host,
                        double *tflops_dfma_host, void *stream);

/* Number of kernel launches this library has enqueued since load (bench.py's gpu_launches). */
long long qmc_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* QMC_B200_H */
