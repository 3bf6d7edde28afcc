/* mtp_b200.h -- C ABI of the B200-native Moment Tensor Potential hot path.
 *
 * What is computed (BASELINE.json north_star; "Inference computes energies,
 * forces, and stresses"; PAPER.md:35,46 configuration-/neighbourhood-mode grades;
 * PAPER.md:62,76 chunked evaluation).  PAPER.md prints no formula; the definitions below
 * restate north_star with the readings G1-G24 listed in DESIGN.md:
 *
 *   r_ij = x_j - x_i + s.H                       (s: image shift, H rows = lattice vectors)
 *   Q_b(r) = T_b(xi(r)) (R_cut - r)^2,  xi = (2r - R_min - R_cut)/(R_cut - R_min), b < n_beta
 *   f_mu(r) = sum_b c[z_i][z_j][mu][b] Q_b(r)
 *   M_{mu,(a,b,c)} = sum_j f_mu(|r_ij|) x^a y^b z^c          (packed symmetric components)
 *   node[dst] += mult * node[src0] * node[src1]              (contraction table, in order)
 *   B_alpha = node[basis_node[alpha]],  E_i = xi0[z_i] + sum_alpha xi[alpha] B_alpha
 *   d_ij = dE_i/dr_ij (reverse pass),  F_k = sum_j d_kj - sum_{i: k in N(i)} d_ik
 *   W_ab = -sum_i sum_j r_ij,a d_ij,b ;  E = sum_i E_i
 *   gamma_i = max_k | sum_alpha B_alpha(n_i) Ainv[alpha][k] |     (neighbourhood mode)
 *   gamma   = max_k | sum_alpha (sum_i B_alpha(n_i)) Ainv[alpha][k] |  (configuration mode)
 *
 * Conventions: every pointer named d_* is a DEVICE pointer owned by the caller; every
 * other pointer is a HOST pointer.  All floating point is IEEE fp64.  Calls enqueue work
 * on `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy default stream) and
 * return without synchronising the host.  Outputs are overwritten, never accumulated.
 * Return value: 0 on success, a negative MTP_E* code otherwise; nothing aborts or throws.
 * There is no CPU fallback: without a CUDA device mtp_create fails with MTP_ECUDA.
 * Threads: a handle carries options, error text and (for the *_host* calls) staging buffers, so one
 * handle serves one host thread at a time; different handles are independent (the compiled contraction
 * kernels are shared through a process-wide cache behind a mutex).  Two calls that use the same workspace
 * must be ordered on the device (same stream, or events).  Exceptions to "return without synchronising":
 * mtp_compute_host, mtp_compute_host_pos, mtp_profile_read, mtp_md_run_al (once per grade evaluation) and
 * the short copies of masses at the start of mtp_md_run.
 */
#ifndef MTP_B200_H
#define MTP_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MTP_OK 0
#define MTP_EINVAL (-1)   /* bad argument / malformed table                              */
#define MTP_ESIZE (-2)    /* workspace too small (see mtp_workspace_bytes)               */
#define MTP_EBOX (-3)     /* d_shift == NULL but a box height is < 2 R_cut               */
#define MTP_ECUDA (-4)    /* CUDA runtime error; text in mtp_last_error                  */
#define MTP_EUNSUP (-5)   /* table outside the compiled kernel family (level > 28, ...)  */
#define MTP_ENOMEM (-6)

typedef struct mtp_handle mtp_handle;

/* Potential description.  HOST pointers, copied at mtp_create.
 * The table fields (basic .. basis_desc) are what mtp_enumerate emits (row a0 of
 * "host-side basis enumerator that emits the contraction table"). */
typedef struct {
  int32_t n_species;        /* S                                                         */
  int32_t n_radial_basis;   /* n_beta (8 in every BASELINE config), 1..16                */
  int32_t n_radial_funcs;   /* n_mu                                                       */
  double r_min, r_cut;      /* Angstrom                                                   */
  int32_t lev_max;          /* informational                                              */
  int32_t n_basic;          /* number of packed moment components                         */
  const int32_t *basic;     /* [n_basic][4] = mu, a, b, c  (a+b+c = nu)                   */
  int32_t n_nodes;          /* n_basic + intermediate components; node k<n_basic = basic k*/
  int32_t n_prod;
  const int32_t *prod;      /* [n_prod][4] = src0, src1, mult, dst; evaluation order;
                               a node is final after the last op that writes it and may
                               only be read after that; dst >= n_basic                    */
  int32_t n_basis;
  const int32_t *basis_node;/* [n_basis] node id of B_alpha, canonical alpha order (G11)  */
  const double *c;          /* [S][S][n_mu][n_beta]  index z_i, z_j, mu, beta (G6)        */
  const double *xi0;        /* [S]                                                        */
  const double *xi;         /* [n_basis]                                                  */
  /* description of each basis function as a multigraph, for cross-checking the order:
     per function: n_components, then per component n_vertices, (mu,nu) per vertex,
     upper-triangular adjacency (row-major).  Ignored by mtp_create; may be NULL.         */
  int32_t n_desc;
  const int32_t *basis_desc;
  const int32_t *basis_desc_off; /* [n_basis+1] offsets into basis_desc                   */
} mtp_params;

/* a0.  Enumerate every scalar contraction with total level <= lev_max (lev(M_{mu,nu}) =
 * 2+4mu+nu; readings G8, G9, G11, G12, G22) and emit the packed-component contraction
 * table.  Fills the table fields of *out (n_radial_funcs, lev_max, n_basic .. basis_desc_off)
 * with malloc'ed arrays; release with mtp_table_free.  lev_max in [2, 28]. */
int mtp_enumerate(int32_t lev_max, mtp_params *out);
void mtp_table_free(mtp_params *table);

/* Create / destroy.  Validates the table (MTP_EINVAL for indices out of range, a node read before its last write,
 * negative multiplicities), turns it into register programs for the contraction kernels (tables whose working set
 * exceeds an SM's registers + shared memory are first cut into a top program and group programs) and compiles them
 * with NVRTC -- seconds of one-time work --, and copies c, xi0, xi to the current CUDA device.  Without libnvrtc
 * the generic table interpreter is set up instead and mtp_last_error(handle) says why. */
int mtp_create(mtp_handle **out, const mtp_params *p);
void mtp_destroy(mtp_handle *h);
const char *mtp_last_error(const mtp_handle *h); /* h may be NULL: last error of a call that
                                                    takes no handle (mtp_create, ..._build_static) */

/* Options (a10 chunk scheduler PAPER.md:62,76; a8 force mode; a12 variant PAPER.md:35). */
#define MTP_OPT_CHUNK_ATOMS 1   /* atoms per chunk ("chunksize"); 0 = automatic: as few equal chunks as
                                   2^20 atoms per chunk and 4 GB of per-atom scratch allow (config 4: one chunk, 4.0 GB
                                   of workspace); smaller chunks trade speed for memory (32 768 atoms: 179 MB)     */
#define MTP_OPT_FORCE_MODE 2    /* MTP_FORCE_GATHER (needs d_rev) | MTP_FORCE_ATOMIC       */
#define MTP_OPT_VARIANT 3       /* MTP_VARIANT_AUTO | _THREAD | _BLOCK                     */
#define MTP_OPT_PROFILE 4       /* 1: record CUDA events around every kernel launch        */
#define MTP_OPT_SKIN_LIST 7     /* 1: the list carries a skin (pairs beyond R_cut; reading G3: they contribute exactly
                                   nothing).  The large-system kernels then first compact every row to its entries within
                                   R_cut (one extra position gather per listed pair) and loop over those only: with a 1 A
                                   skin at R_cut = 5 A that is 1 / 1.73 of the work.  E_i is bit-identical to the default
                                   (0), which multiplies such pairs by zero; forces and virial agree to rounding (their
                                   summation order follows the position in the row) and stay deterministic in gather
                                   mode.  mtp_md_run sets it for skin > 0. */
#define MTP_OPT_CHUNK_PAIRS 6    /* upper bound of the neighbour-list entries of any one chunk: what the per-pair scratch
                                   (packed neighbour words 4 B + d_ij records 32 B per pair) is sized for.  0 = automatic:
                                   1.25 x nnz x chunk_atoms / N + 4096, right for lattice-like inputs; a chunk with more
                                   pairs is counted in MTP_INFO_SCRATCH_OVERFLOW and its excess pairs are dropped.  With a
                                   single chunk the scratch always holds all nnz pairs.                       */
#define MTP_OPT_TREE_CODEGEN 5  /* 1 (default): run the contraction kernels specialised for the table (one register
                                   program per table, generated and compiled with NVRTC at mtp_create);
                                   0: interpret the table with the generic kernel (also what runs when libnvrtc is
                                   absent -- mtp_last_error then says so after mtp_create).  Setting 1 fails with
                                   MTP_EUNSUP when the specialised kernels could not be built.  The two forms sum
                                   in different orders: results agree to rounding, not bit for bit.          */
#define MTP_INFO_TREE_KERNELS 100  /* mtp_get_option only: NVRTC-specialised contraction kernels loaded (0: interpreter) */
#define MTP_INFO_TREE_PROGRAMS 101 /* mtp_get_option only: tables they were built from (1: whole table; else the top
                                      program + the group programs of the partition); kernels = 2 x programs        */
#define MTP_INFO_INPUT_ERRORS 102  /* mtp_get_option only, SYNCHRONISES the device: neighbour-list entries rejected
                                      since the last read (image shift outside {-1,0,1}^3 or index outside [0,N));
                                      such pairs are dropped, so a non-zero count means the results are not valid   */
#define MTP_INFO_SCRATCH_OVERFLOW 103 /* mtp_get_option only, SYNCHRONISES: pairs that did not fit the per-pair scratch of their
                                      chunk since the last read (see MTP_OPT_CHUNK_PAIRS); non-zero = results not valid */
#define MTP_FORCE_GATHER 0      /* deterministic: d_ij kept for one chunk at a time, forces assembled chunk by chunk in
                                   fixed order over the reverse-neighbour index (bit-reproducible run to run)    */
#define MTP_FORCE_ATOMIC 1      /* fp64 atomic scatter; no per-pair scratch              */
#define MTP_FORCE_AUTO 2        /* default: gather when d_rev is given, else atomic      */
#define MTP_VARIANT_AUTO 0
#define MTP_VARIANT_THREAD 1    /* one thread group per atom walks all neighbours (large N) */
#define MTP_VARIANT_BLOCK 2     /* neighbours split across lanes, shuffle-reduced (small N) */
int mtp_set_option(mtp_handle *h, int key, int64_t value);
int mtp_get_option(const mtp_handle *h, int key, int64_t *value);

/* Bytes of device workspace mtp_compute / mtp_grade need for this input size under the
 * current options. */
int mtp_workspace_bytes(const mtp_handle *h, int64_t n_atoms, int64_t nnz, int want_grade,
                        size_t *out_bytes);

/* a1-a8, a10.  Energy, per-atom energy, forces, virial over a full CSR neighbour list.
 *   N <= 2^27 atoms (the kernels pack a neighbour index and its image code into one 32-bit word; MTP_EUNSUP beyond)
 *   d_pos   [N][3] f64      d_type [N] i32 in [0,S)
 *   box     [9] HOST, rows = lattice vectors
 *   d_off   [N+1] i64       d_idx [nnz] i32  (entries with r >= R_cut contribute nothing)
 *   d_shift [nnz][3] i8 image shifts, each component in {-1,0,1} (the kernels pack index and image into one word;
 *           other values are rejected, see MTP_INFO_INPUT_ERRORS), or NULL = minimum image (needs heights > 2 R_cut)
 *   d_rev   [nnz] i32 position of the reverse pair, required in MTP_FORCE_GATHER mode
 *   d_E [1], d_Ei [N] or NULL, d_F [N][3], d_virial [6] = xx,yy,zz,xy,xz,yz (eV) or NULL
 *   d_ws / ws_bytes: scratch of at least mtp_workspace_bytes(...). */
int mtp_compute(mtp_handle *h, int64_t n_atoms, const double *d_pos, const int32_t *d_type,
                const double *box, const int64_t *d_off, const int32_t *d_idx,
                const int8_t *d_shift, const int32_t *d_rev, int64_t nnz, double *d_E,
                double *d_Ei, double *d_F, double *d_virial, void *d_ws, size_t ws_bytes,
                void *cuda_stream);

/* a9.  Extrapolation grades (values are produced only by this call, so
 * there is no stale state as in PAPER.md:100,125).
 *   d_Ainv [n_basis][n_basis] row-major [alpha][k]
 *   mode: 0 neighbourhood (d_gamma_atom [N]), 1 configuration (d_gamma_cfg [1]), 2 both
 *   d_Bsum [n_basis] or NULL: sum_i B(n_i);  d_B [N][n_basis] or NULL: the basis values */
int mtp_grade(mtp_handle *h, int64_t n_atoms, const double *d_pos, const int32_t *d_type,
              const double *box, const int64_t *d_off, const int32_t *d_idx,
              const int8_t *d_shift, int64_t nnz, const double *d_Ainv, int mode,
              double *d_gamma_atom, double *d_gamma_cfg, double *d_Bsum, double *d_B,
              void *d_ws, size_t ws_bytes, void *cuda_stream);

/* Host-buffer convenience path (the end-to-end call bench.py's `e2e` times): same
 * arguments as mtp_compute but every array is a HOST pointer; the library copies them to its own
 * device buffers on a copy stream -- the neighbour list chunk by chunk, so that the evaluation of the
 * first chunks overlaps the transfer of the later ones (pinned host buffers are needed for that
 * overlap) --, runs the same kernels as mtp_compute and copies E, E_i, F, virial back, synchronising
 * before it returns. */
int mtp_compute_host(mtp_handle *h, int64_t n_atoms, const double *pos, const int32_t *type,
                     const double *box, const int64_t *off, const int32_t *idx,
                     const int8_t *shift, const int32_t *rev, int64_t nnz, double *E,
                     double *Ei, double *F, double *virial);

/* Small systems (the "small" GPU variant): one mtp_compute call captured as a CUDA graph and
 * replayed with one launch, which takes the per-kernel launch overhead (a dozen launches of a few microseconds) out of
 * a call that computes for tens of microseconds.  mtp_graph_capture records the call with exactly these buffers --
 * nothing runs yet; mtp_graph_launch enqueues the whole evaluation on the stream: it reads whatever the buffers hold
 * at that time (new coordinates, a list rebuilt in place with the same nnz) and is bit-identical to mtp_compute on
 * the same inputs.  The buffers, the workspace and the handle must outlive the graph; the options of the handle are
 * those at capture time.  Graph launches that overlap on the GPU share the workspace and race. */
typedef struct mtp_graph mtp_graph;
int mtp_graph_capture(mtp_handle *h, int64_t n_atoms, const double *d_pos, const int32_t *d_type, const double *box,
                      const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift, const int32_t *d_rev,
                      int64_t nnz, double *d_E, double *d_Ei, double *d_F, double *d_virial, void *d_ws, size_t ws_bytes,
                      mtp_graph **out);
int mtp_graph_launch(mtp_graph *g, void *cuda_stream);
int mtp_graph_destroy(mtp_graph *g);

/* One rank's share of a sharded evaluation ("full node" runs): the atoms are
 * cut into contiguous ranges, positions and types are replicated, and every rank holds the CSR rows of its own range
 * only.  mtp_compute_rows evaluates the rows [row_lo, row_hi) of an n_atoms system:
 *   d_off [row_hi - row_lo + 1] the window's own CSR (d_off[0] = 0), d_idx / d_shift [nnz] its pairs, d_idx holding
 *   GLOBAL atom indices; d_pos / d_type cover all n_atoms.
 *   d_F [n_atoms][3]: zeroed, then F_i += d_ij and F_j -= d_ij for the window's pairs (fp64 atomics: a window has no
 *   reverse pairs to gather, so MTP_FORCE_GATHER is refused) -- the rank's PARTIAL force on every atom;
 *   d_Ei [n_atoms] or NULL: entries [row_lo, row_hi) are written; d_E, d_virial: the window's partial sums.
 *   Summing d_F, d_E, d_virial over the ranks (one all-reduce of 3 n_atoms + 7 doubles) gives mtp_compute's result
 *   to rounding (the summation order differs).  Workspace: mtp_rows_workspace_bytes(h, n_atoms, n_rows, nnz, 0).
 * mtp_grade_rows: neighbourhood grades of the window (d_gamma_atom [n_atoms], entries of the window written; no
 *   exchange needed) and the window's sum of basis values d_Bsum [n_basis]; the configuration grade follows from the
 *   all-reduced sum through mtp_grade_cfg_from_sum (the GEMV of mtp_grade's mode 1).  Workspace: want_grade = 1. */
int mtp_rows_workspace_bytes(const mtp_handle *h, int64_t n_atoms, int64_t n_rows, int64_t nnz, int want_grade,
                             size_t *out_bytes);
int mtp_compute_rows(mtp_handle *h, int64_t n_atoms, const double *d_pos, const int32_t *d_type, const double *box,
                     int64_t row_lo, int64_t row_hi, const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift,
                     int64_t nnz, double *d_E, double *d_Ei, double *d_F, double *d_virial, void *d_ws, size_t ws_bytes,
                     void *cuda_stream);
int mtp_grade_rows(mtp_handle *h, int64_t n_atoms, const double *d_pos, const int32_t *d_type, const double *box,
                   int64_t row_lo, int64_t row_hi, const int64_t *d_off, const int32_t *d_idx, const int8_t *d_shift,
                   int64_t nnz, const double *d_Ainv, double *d_gamma_atom, double *d_Bsum, void *d_ws, size_t ws_bytes,
                   void *cuda_stream);
int mtp_grade_cfg_from_sum(mtp_handle *h, const double *d_Bsum, const double *d_Ainv, double *d_gamma_cfg,
                           void *cuda_stream);

/* Device neighbour list and MD loop (the paper's rates are atom-timesteps/s of a
 * whole MD step, list builds included; its GPU runs take the list from the host code).
 *
 * mtp_neighbors_build: the full CSR list mtp_compute consumes, from positions and box, on the device.
 *   Listed: every (i, j, s), s in {-1,0,1}^3, (j, s) != (i, 0), with |x_j - x_i + s.H| < r_list (the same operation
 *   order, no contractions); rows ordered by (j, s0, s1, s2) ascending -- bit-identical to a brute-force search over
 *   the 27 images.  Positions should lie in the box; an atom outside is handled as long as no listed shift leaves
 *   {-1,0,1}^3 (such pairs are not listed).
 *   d_off [N+1] i64, d_idx [capacity] i32, d_shift [capacity][3] i8, d_rev [capacity] i32 or NULL (reverse index:
 *   d_rev[p] = position of (j, i, -s)), d_info [2] i64 = { pairs found, errors (rows longer than 256 entries, coordinates that are
 *   not finite) }.
 *   At most `capacity` pairs are written: when d_info[0] > capacity the arrays hold a truncated list (call again
 *   with larger arrays; capacity 0 just counts).  Workspace: mtp_neighbors_workspace_bytes(n_atoms).  No handle: the
 *   list does not depend on the potential.  MTP_EBOX for a singular box. */
int mtp_neighbors_workspace_bytes(int64_t n_atoms, size_t *out_bytes);
int mtp_neighbors_build(int64_t n_atoms, const double *d_pos, const double *box, double r_list, int64_t capacity,
                        int64_t *d_off, int32_t *d_idx, int8_t *d_shift, int32_t *d_rev, int64_t *d_info,
                        void *d_ws, size_t ws_bytes, void *cuda_stream);
/* mtp_neighbors_build_static: mtp_neighbors_build for callers that cannot allocate device memory (code under CUDA
 *   graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same arguments, same kernels and the
 *   same bit-identical result, but no workspace argument: the workspace is a static array in the library's device
 *   image, 6 MiB, which every GPU that loads the library holds until the process exits.  The call itself allocates
 *   nothing (no cudaMalloc / cudaFree, no allocating library routine): it enqueues two memsets and the kernels on
 *   the stream.  Limit: n_atoms <= MTP_NB_STATIC_MAX_ATOMS; beyond it MTP_ESIZE, and mtp_last_error(NULL) names the
 *   limit (use mtp_neighbors_build with your own workspace there).
 *   All calls on a device share the array, which keeps the last call's contents (the call clears what has to start
 *   at zero): calls that overlap on the GPU -- different streams with no ordering between them -- race; calls on
 *   one stream, or ordered by events, are safe.  The first call on each device looks up the array's device address
 *   (cudaGetSymbolAddress): make that first call outside stream capture. */
#define MTP_NB_STATIC_MAX_ATOMS 32768
int mtp_neighbors_build_static(int64_t n_atoms, const double *d_pos, const double *box, double r_list, int64_t capacity,
                               int64_t *d_off, int32_t *d_idx, int8_t *d_shift, int32_t *d_rev, int64_t *d_info,
                               void *cuda_stream);
/* mtp_md_run: n_steps of velocity-Verlet (NVE) with the potential of the handle, entirely enqueued on the stream:
 *   v += dt/2 F/m; x += dt v; [every rebuild_every steps: atoms wrapped into the box, list rebuilt at R_cut + skin];
 *   F = mtp_compute(x); v += dt/2 F/m.   Units: eV, Angstrom, ps, g/mol (LAMMPS "metal"); mass[S] HOST, per species.
 *   d_pos, d_vel are updated in place; d_E[2] = potential and kinetic energy after the last step, d_Ei (or NULL), d_F,
 *   d_virial (or NULL) as mtp_compute returns them for the final positions; d_info[2] = { largest pair count of any
 *   build, accumulated list errors }: the run is valid when d_info[0] <= capacity, d_info[1] == 0 and
 *   MTP_INFO_INPUT_ERRORS / MTP_INFO_SCRATCH_OVERFLOW read 0.  The caller chooses skin and cadence such that no atom
 *   moves more than skin / 2 between builds.  n_steps = 0 evaluates the forces once. */
int mtp_md_workspace_bytes(const mtp_handle *h, int64_t n_atoms, int64_t capacity, size_t *out_bytes);
int mtp_md_run(mtp_handle *h, int64_t n_atoms, double *d_pos, double *d_vel, const int32_t *d_type, const double *box,
               const double *mass, double dt, int64_t n_steps, int32_t rebuild_every, double skin, int64_t capacity,
               double *d_E, double *d_Ei, double *d_F, double *d_virial, int64_t *d_info, void *d_ws, size_t ws_bytes,
               void *cuda_stream);
/* Active-learning policy around the grade: mtp_md_run with the extrapolation grade
 * evaluated on the initial configuration and after every grade_every-th step ("every X timesteps"; 1 = the
 * MLIP-3 style of PAPER.md:106).  mode 0: the largest neighbourhood grade max_i gamma_i (reduced on the device,
 * order independent); mode 1: the configuration grade.  A grade above select_threshold keeps the configuration: its
 * positions go to d_selected[k] (device, [max_selected][N][3], or NULL) and its step and grade to sel_step[k],
 * sel_grade[k] (HOST, [max_selected]) until max_selected are kept.  A grade above break_threshold ends the run after
 * that step ("the simulation is immediately terminated").  The decision is taken on the host: every
 * grade evaluation ends with an 8-byte read and a stream synchronisation; between evaluations the loop only enqueues.
 *   d_Ainv [n_basis][n_basis]; d_gamma_atom [N] or NULL: the neighbourhood grades of the last evaluation (mode 0);
 *   out [4] HOST = { steps done, configurations kept, grade evaluations, 1 when stopped at the break threshold };
 *   max_grade [1] HOST or NULL: the largest grade seen.  Everything else as mtp_md_run.
 * Training / MaxVol selection of the active set stays outside: A^-1 is an input. */
typedef struct mtp_al_policy {
  int32_t grade_every;       /* >= 1 */
  int32_t mode;              /* 0 neighbourhood, 1 configuration */
  double select_threshold;
  double break_threshold;
  int32_t max_selected;      /* >= 0 */
} mtp_al_policy;
int mtp_md_al_workspace_bytes(const mtp_handle *h, int64_t n_atoms, int64_t capacity, size_t *out_bytes);
int mtp_md_run_al(mtp_handle *h, int64_t n_atoms, double *d_pos, double *d_vel, const int32_t *d_type, const double *box,
                  const double *mass, double dt, int64_t n_steps, int32_t rebuild_every, double skin, int64_t capacity,
                  const double *d_Ainv, const mtp_al_policy *policy, double *d_E, double *d_Ei, double *d_F,
                  double *d_virial, int64_t *d_info, double *d_gamma_atom, double *d_selected, int64_t *sel_step,
                  double *sel_grade, int64_t *out, double *max_grade, void *d_ws, size_t ws_bytes, void *cuda_stream);
/* Host positions in, host forces out (what an MD host code does every step): positions and types are copied to the
 * device, the list is built there at R_cut (it never crosses PCIe), the kernels of mtp_compute run in the
 * deterministic force mode, and E, E_i, F, virial are copied back; synchronises.  nnz_out (or NULL): pairs listed. */
int mtp_compute_host_pos(mtp_handle *h, int64_t n_atoms, const double *pos, const int32_t *type, const double *box,
                         double *E, double *Ei, double *F, double *virial, int64_t *nnz_out);

/* Diagnostics (parity bring-up and roofline denominators; not part of the hot path). */
/* Runs K1 + K2 as one chunk and exports the moments M and adjoints G = dE_i/dM, both laid
 * out [n_basic][n_atoms] (component-major), and optionally B [n_atoms][n_basis].  Workspace: the size
 * mtp_workspace_bytes reports with want_grade = 1 and chunk_atoms >= n_atoms. */
int mtp_debug_moments(mtp_handle *h, int64_t n_atoms, const double *d_pos,
                      const int32_t *d_type, const double *box, const int64_t *d_off,
                      const int32_t *d_idx, const int8_t *d_shift, double *d_M, double *d_G,
                      double *d_B, void *d_ws, size_t ws_bytes, void *cuda_stream);
/* With MTP_OPT_PROFILE on: device time (ms, CUDA events on the launching stream) and launch
 * count per kernel class since the last read; classes: 0 moments (K1), 1 tree (K2),
 * 2 pair gradient (K3), 3 force gather, 4 grade (K5).  Synchronises on the recorded events. */
int mtp_profile_read(mtp_handle *h, double *ms /*[5]*/, int64_t *launches /*[5]*/);
/* Host-only (no device needed): how mtp_create will evaluate the contraction table of *p with the specialised
 * kernels (only the table fields are read).  out[8] = { partitioned (0/1), threads (= atoms) per SM of the slowest
 * program, cut rows, groups, ops of the top program, ops summed over the group programs, ops below the cut,
 * specialised (0: more than 120 000 ops after partitioning -- such a table is interpreted) }. */
int mtp_table_plan(const mtp_params *p, int64_t *out);
/* Host-only: the register program of the whole table (kind 0: energy + adjoint, 1: basis values) as data, so that a
 * test can emulate it: prog[cap][7] int32 = op, d, a, b, c, k, x (csrc/tree_codegen.h K2Op), consts[ccap] doubles,
 * info[4] = { instructions, constants, registers, shared-memory slots }.  Only the table fields and xi are read. */
int mtp_k2_program(const mtp_params *p, int kind, int32_t *prog, int64_t cap, double *consts, int64_t ccap,
                   int64_t *info);
/* Number of kernels this library has launched since load (bench.py gpu_launches). */
int64_t mtp_launch_count(void);
/* fp64 FMA throughput microbenchmark: runs `iters` dependent-chain DFMA batches on every
 * SM and returns the useful flop count; time it with CUDA events on `cuda_stream`. */
int mtp_peak_dfma(int64_t iters, double *d_sink, double *out_flops, void *cuda_stream);
/* Algorithmic flops for the roofline report (FMA = 2, each quantity once; formulas in DESIGN.md section 6):
 * flop_per_pair[2] = { K1 moments, K3 pair derivative }, K2 per atom, K5 per atom. */
int mtp_cost_model(const mtp_handle *h, double *flop_per_pair, double *flop_per_atom_tree,
                   double *flop_per_atom_grade);

#ifdef __cplusplus
}
#endif
#endif /* MTP_B200_H */
