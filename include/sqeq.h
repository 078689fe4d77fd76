/* sqeq.h -- C ABI of libsqeq: B200-native periodic Coulomb evaluation for the shadow
 * charge-equilibration MD of arxiv 2503.21176 (cell-list neighbour build, erfc-screened
 * real-space pair sum, smooth Particle Mesh Ewald, and the QEq / shadow-MD drivers built on
 * them).  Citations "PAPER.md:N" are lines of the paper text; "DESIGN.md R-x" are the readings
 * adopted where the paper is silent or garbled.
 *
 * General conventions
 *  - Every call returns SQEQ_OK (0) or a negative SQEQ_E* code; the message is available from
 *    sqeq_last_error(ctx).  No exceptions, no abort().
 *  - "device" pointers are CUDA device memory owned by the caller (e.g. torch tensor
 *    data_ptr()); "host" pointers are ordinary host memory.  The library owns the context, the
 *    neighbour lists, all workspaces and the cuFFT plans.
 *  - All work is enqueued on the context's stream.  A call synchronises that stream only where
 *    it returns a host scalar (documented per call).
 *  - Orthorhombic periodic boxes: box = host double[3] edge lengths (Angstrom).  Positions are
 *    device fp32 [n][3] row-major, any finite values (wrapped internally), |x| < 127 box edges.
 *  - Units: k_e = 1 in sqeq_coulomb (e, Angstrom, e/Angstrom, e^2/Angstrom); the QEq and MD
 *    drivers take ke explicitly (14.3996454784255 eV*Angstrom/e^2 for eV parameters).
 *  - One context per host thread; a context is bound to one device.
 *  - There is no CPU fallback: every entry point fails with SQEQ_ECUDA if no device is usable.
 */
#ifndef SQEQ_H
#define SQEQ_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SQEQ_OK          0
#define SQEQ_EINVAL     -1   /* bad argument (n<=0, box<=0 or non-finite, cutoff>=min(box)/2, rc>list cutoff,
                                grid<order, unsupported order, NULL where not allowed, |x| too large) */
#define SQEQ_ECAPACITY  -2   /* an internal fixed-capacity buffer overflowed (message says which) */
#define SQEQ_ECUDA      -3   /* CUDA runtime error */
#define SQEQ_ECUFFT     -4   /* cuFFT error */
#define SQEQ_ENOTCONV   -5   /* sqeq_qeq_solve: max_iter reached; last iterate and residual still written */
#define SQEQ_ENOMEM     -6   /* device or host allocation failed */

typedef struct sqeq_ctx   sqeq_ctx;    /* opaque: stream, workspaces, cuFFT plans */
typedef struct sqeq_nlist sqeq_nlist;  /* opaque: device neighbour list + cell-major permutation */

/* ---- context ------------------------------------------------------------------------------- */
/* device: CUDA ordinal.  cuda_stream: a cudaStream_t (may be NULL = legacy default stream); the
 * caller keeps ownership of the stream. */
int  sqeq_create (sqeq_ctx** out, int device, void* cuda_stream);
/* Synchronises, releases everything the context owns -- including the device storage of neighbour lists that
 * are still alive: their handles stay valid for sqeq_nl_free / sqeq_nl_count only. */
int  sqeq_destroy(sqeq_ctx* ctx);
/* Context-owned NUL-terminated message of the last failing call; never freed by the caller.
 * ctx may be NULL (returns the message of the last failing sqeq_create in this thread). */
const char* sqeq_last_error(const sqeq_ctx* ctx);
/* Library version string and the compute capability it was built for ("sm_100a"). */
const char* sqeq_version(void);

/* ---- neighbour list: PAPER.md:43-71 (section 3.1, Alg. 1) ------------------------------------
 * Builds the list of all pairs with minimum-image distance STRICTLY below `cutoff`
 * (= r_c + skin), defined as the fp64 predicate of DESIGN.md R-NL evaluated on the fp32 input
 * values, so the set is unique and bit-reproducible.
 *   n       number of atoms, 1 <= n < 2^27
 *   pos     device fp32 [n][3]
 *   box     host double[3]
 *   cutoff  list cutoff; must satisfy 0 < cutoff < min(box)/2 (one image per pair)
 *   out     receives a new list handle (free with sqeq_nl_free)
 * Internally: atoms are wrapped, binned into cells of edge >= cutoff/2, reordered cell-major; the
 * list is directed rows over the reordered atoms, entries either 16-bit indices into the neighbourhood
 * of the atom's 2x2x2 cell group or 32-bit (atom index | 27-valued image code).  Synchronises the
 * stream (the pair count sizes the list allocation).  SQEQ_ECAPACITY if an atom has more neighbours
 * than the per-warp staging rows in shared memory hold (about 12,700 in the 16-bit format, 6,300 in the 32-bit
 * one). */
int  sqeq_nl_build (sqeq_ctx* ctx, int64_t n, const float* pos, const double box[3],
                    double cutoff, sqeq_nlist** out);
/* Number of unique (i<j) pairs in the list.  host int64 out. */
int  sqeq_nl_count (const sqeq_nlist* nl, int64_t* n_pairs_unique);
/* Canonical export for parity: unique pairs i<j in the CALLER's atom numbering, sorted by (i,j);
 * shift3[k] = int8[3] s such that pos[j] + s*box - pos[i] (raw, unwrapped caller positions at
 * build time) is the in-range vector.  i, j: device int32 [n_pairs_unique]; shift3: device int8
 * [n_pairs_unique][3]; caller-owned.  Synchronises the stream. */
int  sqeq_nl_export(sqeq_ctx* ctx, const sqeq_nlist* nl, int32_t* i, int32_t* j, int8_t* shift3);
/* The paper's two output formats, DIRECTED rows in the caller's numbering, neighbours of an atom in
 * ascending order, shift = image shift of the ordered pair (i, j) on the raw caller positions at build time:
 *   ELLPACK: nbr device int32 [n][K], row i = the neighbours of atom i padded with -1; shift3 device int8 [n][K][3];
 *            counts device int32 [n] (may be NULL) = neighbours per atom.  K >= the longest row (sqeq_nl_info), else
 *            SQEQ_ECAPACITY.
 *   COO:     i, j device int32 [2 * n_pairs_unique], shift3 device int8 [..][3]: every pair in both directions,
 *            sorted by (i, j).
 * Both synchronise the stream. */
int  sqeq_nl_export_ellpack(sqeq_ctx* ctx, const sqeq_nlist* nl, int K, int32_t* nbr, int8_t* shift3, int32_t* counts);
int  sqeq_nl_export_coo(sqeq_ctx* ctx, const sqeq_nlist* nl, int32_t* i, int32_t* j, int8_t* shift3);
/* List introspection (host outputs, any may be NULL): cells per axis, directed entries, max row. */
int  sqeq_nl_info  (const sqeq_nlist* nl, int ncell[3], int64_t* n_directed, int* max_row);
/* Bytes per stored list entry: 2 (16-bit index into the cell group's neighbourhood, the format of the
 * shared-memory-staged real-space kernel) or 4 (atom index | image code; used when a neighbourhood
 * does not fit 16 bits / shared memory). */
int  sqeq_nl_entry_bytes(const sqeq_nlist* nl, int* bytes);
/* Storage layout of a built list (host outputs, any may be NULL).  n_slots: list slots in use -- the 16-bit
 * format pads every row to a multiple of 32 slots (padding entries point at a far-away dummy atom), so
 * n_slots >= directed entries (it also counts the unused tail of each cell group's reserved slice).  entry_shift: a 16-bit entry is (local index << entry_shift); 4 (byte offset
 * of a 16-byte staged atom) while the most populous neighbourhood stays below 4095 atoms, else 0.
 * max_neighbourhood: atoms (all periodic images) the staged real-space kernel holds per cell group. */
int  sqeq_nl_layout(const sqeq_nlist* nl, int64_t* n_slots, int* entry_shift, int* max_neighbourhood);
/* Largest distance (Angstrom, host double) any atom has moved since the list was built, from the caller's
 * positions pos[n][3] (device) and the copy the list keeps of the positions it was built from.  A list built
 * with cutoff rc + skin holds every pair with r < rc while this stays below skin/2: rebuild
 * when it does not.  One small kernel and a stream synchronisation; +inf if a position is NaN. */
int  sqeq_nl_max_drift(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, double* max_drift);
/* The same for the positions pos + dt * vel (vel: device fp32 [n][3]): what the drift will be after the position
 * update of the next MD step (up to its dt^2 a/2 term, ~0.01 Angstrom for water at 0.5 fs).  An MD loop rebuilds
 * BEFORE a step whenever this reaches skin/2 minus that slack, so that no evaluation ever runs on a list that is
 * no longer complete ("rebuilt when the maximum displacement exceeds half the skin"). */
int  sqeq_nl_max_drift_ahead(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const float* vel,
                             double dt, double* max_drift);
int  sqeq_nl_free  (sqeq_nlist* nl);

/* ---- Coulomb evaluation: Eq. 2 = Eq. 3 (real space, r < rc) + Alg. 2 (smooth PME,
 * PAPER.md:140-151) + Eq. 5 (self term) ------------------------------------------------------
 *   nl      list built from (an earlier state of) these atoms; positions may have moved by less
 *           than (list cutoff - rc)/2 since the build.  Pairs are re-tested against rc in-kernel.
 *   pos     device fp32 [n][3], current positions, caller order
 *   q       device fp32 [n], charges (any vector: Krylov vectors need not be neutral; the uniform
 *           background term is omitted, DESIGN.md R-G11)
 *   rc      real-space cutoff, 0 < rc <= list cutoff
 *   alpha   Ewald splitting parameter (1/Angstrom), > 0
 *   grid    host int[3] PME grid points per axis, each >= order and even; order in 4..8 (6 is the paper's; for the odd ones
 *           the Nyquist plane is left out of the influence function, reading G19)
 *   phi     device fp32 [n]    out: phi_i = dE/dq_i (may be NULL)
 *   force   device fp32 [n][3] out: F_i = -dE/dr_i; NULL selects the cheaper potential-only mode
 *   energy  host double* out: E = 1/2 sum q_i phi_i (may be NULL; non-NULL synchronises the stream)
 */
int  sqeq_coulomb  (sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                    const float* q, const double box[3], double rc, double alpha,
                    const int grid[3], int order, float* phi, float* force, double* energy);

/* The same evaluation without any synchronisation: everything, including the fp64 reduction of
 * E = 1/2 sum q_i phi_i when want_energy != 0, is enqueued on the context's stream and the call
 * returns.  The energy stays in a context-owned device scalar until sqeq_energy_fetch copies the
 * value of the LAST enqueued evaluation to the host (that call synchronises the stream).  For
 * callers that step many evaluations back to back (MD, Krylov loops) and read energies rarely. */
int  sqeq_coulomb_enqueue(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                          const float* q, const double box[3], double rc, double alpha,
                          const int grid[3], int order, float* phi, float* force, int want_energy);
int  sqeq_energy_fetch(sqeq_ctx* ctx, double* energy);

/* The same evaluation with HOST buffers (pos, q, phi, force are host fp32 arrays, ideally pinned):
 * host->device copies of pos and q, the evaluation, and device->host copies of phi / force all
 * happen inside the call on the context's stream; always synchronises.  This is the end-to-end
 * entry bench.py times (copies inside the timed region). */
int  sqeq_coulomb_host(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos_host,
                       const float* q_host, const double box[3], double rc, double alpha,
                       const int grid[3], int order, float* phi_host, float* force_host,
                       double* energy);

/* The same evaluation, PIPELINED for independent evaluations: submit enqueues the host->device copies on a copy
 * stream, the evaluation on the context's stream and the device->host copies on a second copy stream, and
 * returns without synchronising; wait blocks until the results of that slot are in phi_host / force_host
 * (and returns the energy if it was asked for at submit).  Two slots (0, 1): while slot s computes, the inputs
 * of the other slot travel in and its previous results travel out.  Host buffers must be pinned and stay
 * untouched between submit and wait; a slot cannot be submitted again before it was waited for (EINVAL).
 * The neighbour list may be freed after submit (its storage is released in stream order). */
int  sqeq_coulomb_host_submit(sqeq_ctx* ctx, int slot, const sqeq_nlist* nl, int64_t n,
                              const float* pos_host, const float* q_host, const double box[3],
                              double rc, double alpha, const int grid[3], int order,
                              float* phi_host, float* force_host, int want_energy);
int  sqeq_coulomb_host_wait(sqeq_ctx* ctx, int slot, double* energy);

/* ---- regular Ewald summation: PAPER.md:98-132 (section 3.2, Eqs. 6-12); SURVEY.md 8(f) NEXT-3 ---------------
 * The same evaluation with the reciprocal part summed directly over the k-vectors k = 2 pi (m_x/L_x, m_y/L_y,
 * m_z/L_z), m != 0, |m_d| <= kmax[d] (host int[3], each in [1, 128]) instead of on a mesh: the structure
 * factors S(k) = sum_i q_i e^{i k.r_i} (Eqs. 7-9), then Eqs. 10-11 per atom, the phase matrix of Eq. 9 formed
 * block by block on the fly and never stored.  O(N * number of k-vectors): the faster method below about 5,000
 * atoms.  Real-space part, self term, arguments and outputs as for sqeq_coulomb.  A non-NULL
 * energy synchronises. */
int  sqeq_coulomb_ewald(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const float* q,
                        const double box[3], double rc, double alpha, const int kmax[3], float* phi,
                        float* force, double* energy);
/* Parameters from an accuracy delta by the heuristics the paper takes from OpenMM (the formulas
 * are that library's, recalled -- DESIGN.md reading G17): alpha = sqrt(-ln 2 delta)/rc; kmax[d] for
 * sqeq_coulomb_ewald; grid[d] = ceil(2 alpha L_d/(3 delta^(1/5))) rounded up to an even 2^a 3^b 5^c for
 * sqeq_coulomb.  Host outputs, any may be NULL.  No context needed. */
int  sqeq_ewald_params(const double box[3], double rc, double delta, double* alpha, int kmax[3], int grid[3]);

/* ---- fixed geometry, many charge vectors ("Each iteration involves
 * calculating a Coulomb-like potential") ------------------------------------------------------
 * Every Krylov iteration of a QEq solve and all 2 + m evaluations of a shadow-MD step repeat the evaluation on
 * the SAME positions with another charge vector.  sqeq_geometry_set prepares the positions once (re-gather,
 * fractional grid coordinates; arguments as for sqeq_coulomb); each sqeq_coulomb_fixed then evaluates one
 * charge vector q (device fp32 [n]) on them.  The first evaluation also writes the GEOMETRY CACHE -- per row
 * of the list the entries with r < rc and their erfc(alpha r)/r (and the field factor when forces are asked
 * for) -- and the later ones run the real-space part as a sparse product over it: no erfc/exp/rsqrt, no skin
 * entries (10 B per list slot of device memory, owned by the context).  phi may be NULL when force is given
 * (field only).  The cache is dropped by any other evaluation or neighbour build on the context.  No
 * synchronisation; the energy, if asked for, is read with sqeq_energy_fetch.  sqeq_qeq_solve and
 * sqeq_shadow_md_* use the same mechanism internally. */
int  sqeq_geometry_set (sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const double box[3],
                        double rc, double alpha, const int grid[3], int order);
int  sqeq_coulomb_fixed(sqeq_ctx* ctx, int64_t n, const float* q, float* phi, float* force, int want_energy);
/* The batched form (the other half of NEXT-1): potentials of nvec (1..64) charge vectors q[nvec][n]
 * (device fp32, row v = vector v) on the geometry of the last sqeq_geometry_set -> phi[nvec][n].  Up to four vectors
 * share ONE pass over the geometry cache for the real-space part (the cache stream bounds the single-vector kernel:
 * 0.145 ms for one vector at 331,776 atoms, 0.19 for four); the reciprocal part runs per vector on the shared prepared
 * geometry.  The first vector on a fresh geometry is evaluated alone (it writes the cache).  No synchronisation. */
int  sqeq_coulomb_fixed_batch(sqeq_ctx* ctx, int64_t n, int nvec, const float* q, float* phi);

/* Parts of the last sqeq_coulomb call on this context, for diagnostics and stage-wise parity
 * (caller order; device fp32 outputs, any may be NULL): phi_real[n], F_real[n][3], phi_rec[n],
 * F_rec[n][3]; host double E_rec = 1/2 sum_m G|Qhat|^2 (Alg. 2 step 3).  Synchronises. */
int  sqeq_coulomb_parts(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, float* phi_real,
                        float* F_real, float* phi_rec, float* F_rec, double* E_rec);
/* Copies the PME real-space grids of the last call: charge grid Q after step 1 (if which = 0) or
 * potential grid Phi after step 4 (which = 1) into device fp32 out[K0][K1][K2]. */
int  sqeq_pme_grid (sqeq_ctx* ctx, int which, float* out);

/* ---- QEq solve: Eq. 18, matrix-free GMRES with C v = J o v + ke*phi[v]
 * (PAPER.md:186-194); zero initial guess, fp64 Krylov basis, CGS2 orthogonalisation --------------
 *   chi, J      device fp32 [n] electronegativity and hardness
 *   tol         stop when the GMRES residual estimate ||b-Ax||/||b|| <= tol
 *   max_iter    maximum number of Coulomb evaluations; restart: Krylov dimension (0 = unrestarted,
 *               i.e. up to max_iter vectors)
 *   q_out       device fp32 [n]; lambda_out, iters_out, relres_out: host scalars (may be NULL).  *iters_out counts the
 *               Coulomb evaluations the returned solution is built from; with tol > 0 the host judges an iteration
 *               while the next one already runs, so one further evaluation is launched and discarded
 * Returns SQEQ_ENOTCONV if tol was not reached (outputs are still written).  Synchronises. */
int  sqeq_qeq_solve(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                    const double box[3], double rc, double alpha, const int grid[3], int order,
                    double ke, const float* chi, const float* J, double total_charge,
                    double tol, int max_iter, int restart,
                    float* q_out, double* lambda_out, int* iters_out, double* relres_out);
/* The same solve with the options the paper's regular-MD runs use: jacobi != 0 applies the right
 * Jacobi preconditioner diag(J_i + ke A_ii) (A_ii: the Ewald self-image diagonal; 1 on the constraint row);
 * q0 != NULL (device fp32 [n]) and lambda0 give the initial guess (its residual costs one evaluation). */
int  sqeq_qeq_solve_pc(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                       const double box[3], double rc, double alpha, const int grid[3], int order,
                       double ke, const float* chi, const float* J, double total_charge,
                       double tol, int max_iter, int restart, int jacobi, const float* q0, double lambda0,
                       float* q_out, double* lambda_out, int* iters_out, double* relres_out);

/* ---- shadow XL-BOMD step: PAPER.md:196-246 (Eqs. 19-27); DESIGN.md R-MD -------------------------
 * State arrays are caller-owned device memory, updated in place:
 *   pos [n][3], vel [n][3] fp32 (Angstrom, Angstrom/fs); mass [n] fp32 (amu);
 *   nhist fp64 [7][n]: rows 0..5 = n(t), n(t-dt), ..., n(t-5dt) (most recent first),
 *                      row 6 = dt^2 * ndd(t), the solution of Eq. 27 at the current time level;
 *   chi, u [n] fp32 (eV/e, eV/e^2);
 *   force [n][3] fp32: F(t) = -grad U(R, n) of Eq. 21/25 (eV/Angstrom), in and out.
 *   V_short stand-in: atoms 3m, 3m+1, 3m+2 form O,H,H with harmonic O-H and H-H terms
 *   (k_oh, r_oh, k_hh, r_hh; eV/Angstrom^2, Angstrom); pass k_oh = k_hh = 0 to disable.
 * sqeq_shadow_md_init: sets the history and evaluates force, row 6 and energies at t = 0.
 *   max_iter > 0: n(0) = q_min from sqeq_qeq_solve(tol, max_iter, unrestarted), copied to rows 0..5
 *                 (returns SQEQ_ENOTCONV if tol is not reached);
 *   max_iter = 0: the caller supplies n(0) in row 0; it is copied to rows 1..5.
 * sqeq_shadow_md_step: one velocity-Verlet step of length dt (fs) for R and one Verlet step with
 *   dissipation for n,  n(t+dt) = 2n(t) - n(t-dt) + dt^2 ndd(t) + alpha_diss sum_k c_k n(t-k dt),
 *   then, at t+dt: v = ke*phi[n], q[n] from Eq. 22, forces, and `krylov_rank` GMRES steps (zero
 *   start) on Eq. 27, J x = -kappa (q[n]-n) with kappa = dt^2 omega^2 (krylov_rank = 0: J ~ -I).
 *   Coulomb evaluations per step: 2 (potential+field of n, field of q-n) + krylov_rank.
 *   The list may be stale by less than (list cutoff - rc)/2, as for sqeq_coulomb.
 * energies: host double[4] out = {shadow potential energy U (Eq. 20/21 incl. stand-in), kinetic
 * energy (0 from init), ||q[n]-n||_2, Coulomb evaluations done}; may be NULL (then the call does
 * not synchronise, except inside the Krylov iterations). */
typedef struct sqeq_md_params {
    double dt;            /* fs */
    double ke;            /* eV*Angstrom/e^2 */
    double total_charge;
    double rc, alpha;
    int    grid[3];
    int    order;
    int    krylov_rank;   /* m Krylov updates per step (cfg 4: 4) */
    double k_oh, r_oh, k_hh, r_hh;
    double kappa;         /* dt^2 omega^2 */
    double alpha_diss;    /* dissipation strength */
    double c[7];          /* dissipation coefficients c_0..c_5 (c[6] unused) */
    double krylov_tol;    /* > 0: solve Eq. 27 to this relative residual (Table 1's "Sol. Tol.")
                             with at most krylov_rank vectors (one host synchronisation per vector); 0: exactly
                             krylov_rank vectors, no synchronisation */
    double k_rep, r_rep;  /* V_short stand-in, second part: soft-sphere repulsion 1/2 k_rep (r_rep - r)^2 between the
                             oxygens (atoms 3m) of different molecules for r < r_rep (eV/Angstrom^2, Angstrom); it
                             plays the part of the O-O Lennard-Jones term of three-site water models.  k_rep = 0
                             disables it.  Needs r_rep + (list cutoff - rc) <= the list's cell edge (>= cutoff/2). */
} sqeq_md_params;

int  sqeq_shadow_md_init(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                         const double box[3], const sqeq_md_params* p, const float* chi,
                         const float* u, double tol, int max_iter,
                         double* nhist, float* force, double* energies);
int  sqeq_shadow_md_step(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, float* pos, float* vel,
                         const float* mass, const double box[3], const sqeq_md_params* p,
                         const float* chi, const float* u, double* nhist, float* force,
                         double* energies);

/* nsteps shadow-MD steps in one call, the neighbour list kept valid by the library: it is rebuilt (cutoff
 * list_cutoff = rc + skin, which must be the cutoff of *nl_io) before a step whenever the largest displacement since
 * the build would reach skin/2 - slack, judged WITHOUT waiting for the GPU each step: the test looks
 * two steps ahead from a number the device reduced two steps ago (the first steps after a build are checked
 * synchronously).  slack (Angstrom) covers the 2 dt^2 a of that extrapolation: 0.05 for water at 0.5 fs.
 * *nl_io: in, a list built for the current positions; out, the list in use at the end (the caller frees it; lists
 * replaced on the way are freed by the call).  stats: host double[8] out = {U, kinetic energy, |q[n]-n|, Coulomb
 * evaluations of the last step, rebuilds, largest look-ahead displacement accepted, displacement at the end,
 * skin/2}; may be NULL.  Synchronises at the end (and at every rebuild). */
int  sqeq_shadow_md_run(sqeq_ctx* ctx, sqeq_nlist** nl_io, int64_t n, float* pos, float* vel, const float* mass,
                        const double box[3], const sqeq_md_params* p, const float* chi, const float* u,
                        double* nhist, float* force, int nsteps, double list_cutoff, double slack, double* stats);

/* ---- regular Born-Oppenheimer MD: PAPER.md:155-200 (Eqs. 13-19), the method shadow MD is compared with
 * (Table 1, 321-323) -------------------------------------------------------------------
 * Every step solves Eq. 18 for q_min by GMRES to the relative residual `tol` (at most max_iter Coulomb
 * evaluations; jacobi != 0: right Jacobi preconditioner diag(u_i + ke A_ii); warm_start != 0: the
 * previous step's charges and lambda are the initial guess, whose residual costs one evaluation), then
 * evaluates F = ke F_Coul[q_min] + stand-in at FIXED charges (Eq. 19) and U_BO (Eq. 28).
 * State, caller-owned device memory: pos, vel [n][3] fp32; q fp64 [n] (charges, in and out); force [n][3] fp32;
 * lambda: host double, in and out.  p->krylov_rank, kappa, alpha_diss, c are not used.
 * energies: host double[4] out = {U_BO, kinetic energy (0 from init), relative residual reached, Coulomb
 * evaluations = solver evaluations + 1}.  Both calls synchronise.  SQEQ_ENOTCONV if tol is not reached
 * (state and energies are still written). */
int  sqeq_bomd_init(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const double box[3],
                    const sqeq_md_params* p, const float* chi, const float* u, double tol, int max_iter,
                    int jacobi, double* q, double* lambda, float* force, double* energies);
int  sqeq_bomd_step(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, float* pos, float* vel, const float* mass,
                    const double box[3], const sqeq_md_params* p, const float* chi, const float* u, double tol,
                    int max_iter, int jacobi, int warm_start, double* q, double* lambda, float* force,
                    double* energies);

/* ---- per-stage device timing (CUDA events on the context's stream) ----------------------------
 * Stages: see SQEQ_T_*.  Enable, run, then read: total milliseconds and number of launches per
 * stage since the last reset.  sqeq_profile_read synchronises the stream. */
enum {
    SQEQ_T_NL_BIN = 0,   /* bin + sort + reorder                      (a-1) */
    SQEQ_T_NL_PAIRS,     /* pair enumeration, count + fill            (a-2) */
    SQEQ_T_PREP,         /* per-evaluation re-gather / fractional coordinates */
    SQEQ_T_REAL,         /* real-space erfc pair sum                  (a-3) */
    SQEQ_T_SPREAD,       /* B-spline spreading incl. grid clear       (a-4) */
    SQEQ_T_FFT_FWD,      /* forward transforms but the x pass         (a-5) */
    SQEQ_T_INFLUENCE,    /* influence multiply + energy               (a-6) */
    SQEQ_T_FFT_INV,      /* inverse transforms but the x pass         (a-7) */
    SQEQ_T_GATHER,       /* gather                                    (a-8) */
    SQEQ_T_ASSEMBLE,     /* self term, sum, un-permute, energy        (a-9) */
    SQEQ_T_KRYLOV,       /* GMRES / MD vector algebra                 (a-10, a-11) */
    SQEQ_T_COUNT
};
int  sqeq_profile_enable(sqeq_ctx* ctx, int on);
int  sqeq_profile_reset (sqeq_ctx* ctx);
int  sqeq_profile_read  (sqeq_ctx* ctx, int stage, double* total_ms, int64_t* launches);
/* Switches (also read from the environment by sqeq_create, as SQEQ_<NAME IN CAPITALS>=0/1):
 *   "graphs"           1  replay launch-bound sequences (sqeq_coulomb_fixed on a cached geometry, the steps of
 *                         sqeq_shadow_md_run) as CUDA graphs; needs a context stream other than the legacy default
 *   "overlap"          1  PME on an internal side stream beside a persistent real-space grid: 0 never, 1 for
 *                         force evaluations the caller does not wait for (sqeq_coulomb_enqueue, sqeq_coulomb with
 *                         energy == NULL, sqeq_coulomb_host_submit: +3 % throughput at 331,776 atoms, +14 % at 98,304),
 *                         2 always (a single evaluation that is waited for finishes LATER that way, and a potential-
 *                         only one takes 0.47 instead of 0.40 ms at 331,776 atoms)
 *   "real_lean_blocks" 2  blocks per SM of that persistent grid
 *   "fft_fused"        1  x-axis transforms fused with the influence multiply in one own kernel between batched 2-D
 *                         cuFFT transforms (0, or a grid whose x size has a prime factor above 5: 3-D cuFFT transforms
 *                         and a separate influence kernel)
 *   "fft_xline2"       1  that kernel in its register-resident form (two small DFTs around one shared-memory exchange
 *                         per transform) for x sizes 24, 32, 48, 64, 72, 80, 96, 108, 120, 128, 144, 160, 192, 256; 0 or
 *                         another size: radix-2/3/4/5 passes through shared memory
 *   "fft_own"          1  the y and z passes by own kernels of the same kind too (no cuFFT call in an evaluation) when all
 *                         three extents are among those sizes; 0: batched 2-D cuFFT transforms over (y, z)
 *   "pme_atom_sched"   1  in those kernels, atoms dealt to lanes by the shared-memory bank their footprint starts on (a warp's
 *                         lanes then never collide): 0 never, 1 from four tiles per SM on (-8 us at 331,776 atoms), 2 always
 *   "pdl"              1  the transform kernels are launched with programmatic stream serialisation (each starts its
 *                         prologue while the one before drains and waits, griddepcontrol.wait, before touching data):
 *                         -2 us per evaluation where the five kernels are not hidden behind the real-space kernel
 *   "pairs_staged"     1  pair enumeration with the cell group's neighbourhood staged in shared memory (from the second
 *                         build of a system on, when the neighbourhood size is known); 0: always the segment sweep
 *   "real_tma"         0  geometry-cache rows streamed into shared memory by the bulk-copy engine (cp.async.bulk +
 *                         mbarrier, two rows in flight per warp) instead of per-lane vector loads; 4 % slower at
 *                         331,776 atoms (0.151 vs 0.145 ms), kept as the measured alternative
 *   "pme_atom_threads" 1  one thread per atom in the tile kernels (a third of the instructions of the lane-group
 *                         mapping): 0 never, 1 when the grid has at least two tiles per SM, 2 always
 *   "pme_tiles"        1  shared-memory tiles for spreading and gathering (0: global-memory kernels)
 *   "spread_float"     0  fp32 compare-and-swap accumulation in the spreading tile instead of fixed point
 *   "real_staged"      1  16-bit list + shared-memory-staged real-space kernel (0: 32-bit list, global gather;
 *                         takes effect at the next sqeq_nl_build)
 * Synchronises the stream.  SQEQ_EINVAL for an unknown name. */
int  sqeq_set_option(sqeq_ctx* ctx, const char* name, int value);
/* ---- an entry point that allocates nothing --------------------------------------------------------------------
 * E = 1/2 sum_i q_i phi_i (Eq. 5; what sqeq_coulomb returns in *energy, k_e = 1) for callers that cannot
 * call cudaMalloc (CUDA-graph capture, serving loops, harnesses that forbid it): no context, no cudaMalloc / cudaFree,
 * no allocating library routine.  The reduction's scratch (one fp64 partial sum per 1,024 atoms and a counter) is a
 * file-scope __device__ array of 32.25 KB that every GPU loading the library holds until exit; hence the limit
 * n <= SQEQ_NOALLOC_MAX_N, beyond which the call returns SQEQ_EINVAL with a message in sqeq_last_error(NULL).
 *   device      ordinal; made current.  cuda_stream: cudaStream_t (may be 0); the work is enqueued there, no
 *               synchronisation.  The first call per device looks up the array's device address (not under capture).
 *   q, phi      device fp32 [n], caller-owned;  energy_dev: DEVICE double, written when the kernel runs
 * All calls on a device share the array: calls that overlap on the GPU (different streams) race; calls on one stream
 * are ordered.  Fixed summation order: the same inputs give the same bits on every call. */
#define SQEQ_NOALLOC_MAX_N 4194304
int  sqeq_energy_noalloc(int device, void* cuda_stream, int64_t n, const float* q, const float* phi, double* energy_dev);

/* Number of the library's own kernel launches (cuFFT's excluded) since sqeq_create / last reset. */
int  sqeq_launch_count  (sqeq_ctx* ctx, int64_t* launches, int reset);

#ifdef __cplusplus
}
#endif
#endif /* SQEQ_H */
