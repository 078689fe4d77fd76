// common.cuh -- internal declarations of libsqeq (context, list, error and timing helpers).
// Not part of the public boundary (include/sqeq.h is).
#pragma once
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <functional>
#include <vector>

#include "../../include/sqeq.h"
#include "cellgroup.cuh"

#define SQEQ_MAX_ORDER 8
#define SQEQ_NHIST 7
#define REAL_STAGE_MAX_BYTES (160 * 1024)   // staged neighbourhood of the real-space kernel

struct DevBuf {
    void*  p = nullptr;
    size_t cap = 0;
};

struct sqeq_nlist;

struct TimerRec {
    int stage;
    cudaEvent_t a, b;
};

// NEXT-1 geometry cache of the real-space sum (realspace.cu): per row of the list, the entries with r < rc and
// their t = erfc(alpha r)/r (and g), valid for (list, positions of the last prep_atoms, rc, alpha)
enum { GEOM_NEW = 0, GEOM_FIXED = 1 };
struct GeomCache {
    bool valid = false;
    const sqeq_nlist* nl = nullptr;
    uint64_t serial = 0;
    double rc = 0, alpha = 0;
    DevBuf idx, t, len;
};

struct sqeq_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    cudaStream_t stream2 = nullptr;       // side stream: PME runs beside the real-space kernel
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    char err[512] = {0};
    int sm_count = 148;
    cudaMemPool_t pool = nullptr;         // stream-ordered pool for neighbour-list storage (kept across rebuilds)
    double* h_kry = nullptr;              // pinned: GMRES coefficients of a whole cycle (deferred host pass)
    size_t h_kry_cap = 0;
    cudaEvent_t kry_ev[4] = {nullptr, nullptr, nullptr, nullptr};   // behind the coefficient copies of the last iterations
    int64_t nl_last_n = 0, nl_last_total = 0;   // sizes of the previous build: next build's estimate
    int nl_last_max_row = 0;
    int nl_last_fmt = 1;
    int nl_last_max_pop = 0;
    int64_t nl_last_pairs = 0;
    bool spread_float = false;            // SQEQ_SPREAD_FLOAT=1: fp32 (CAS) instead of fixed-point shared accumulation
    int overlap = 1;                      // "overlap": 0 never, 1 (default) evaluations nobody waits for, 2 always: PME on
                                          // the side stream beside a persistent real-space grid
    bool throughput_call = false;         // set by the entry point: the caller does not wait for this evaluation
    bool overlap_now = false;             // decision of the evaluation being enqueued (coulomb_eval)
    int real_lean_blocks = 2;             // SQEQ_REAL_LEAN_BLOCKS: persistent real-space blocks per SM with SQEQ_OVERLAP=1
    bool real_tma = false;                // "real_tma": geometry-cache rows streamed with cp.async.bulk + mbarrier (measured
                                          // 4 % slower than per-lane vector loads at cfg 4: an option)
    bool pairs_staged_off = false;        // "pairs_staged" = 0: always the segment-sweep pair kernel (k_pairs)
    bool real_staged_off = false;         // SQEQ_REAL_STAGED=0: 32-bit list + global-gather real-space kernel

    // ---- PME state (cached by grid/order/box/alpha) ----
    int K[3] = {0, 0, 0};
    int order = 0;
    double tab_box[3] = {0, 0, 0};
    double tab_alpha = 0;
    cufftHandle plan_r2c = 0, plan_c2r = 0;
    bool plans_ok = false;
    // fused x-axis pass (pme.cu, k_xline_influence): batched 2-D plans over (y,z), twiddles, radix schedule
    cufftHandle plan2_r2c = 0, plan2_c2r = 0;
    bool xf_ok = false;
    bool fft_fused_off = false;           // SQEQ_FFT_FUSED=0: 3-D cuFFT transforms + separate influence kernel
    bool pdl_off = false;                 // "pdl" = 0: ordinary stream-ordered launches everywhere
    bool fft3_ok = false;                 // all three grid extents are sizes fftx.cu / fftz.cu are built for
    bool fft_own_off = false;             // "fft_own" = 0: cuFFT for the y and z axes even then
    bool fft_xline2_off = false;          // "fft_xline2" = 0: the Stockham x-pass (pme.cu) even where fftx.cu has the size
    int xf_npass = 0, xf_radix[12] = {0};
    DevBuf xf_tw;
    int pme_atom_threads = 1;             // "pme_atom_threads": one thread per atom in the tile kernels: 0 never (lane
                                          // groups), 1 when there are at least two tiles per SM, 2 always
    int pme_atom_sched = 1;               // "pme_atom_sched": lanes dealt by start bank in those kernels: 0 never, 1 from four
                                          // tiles per SM on, 2 always
    bool pme_tiles_off = false;           // SQEQ_PME_TILES=0: global-memory spread/gather only (testing)
    DevBuf grid;      // float  [K0][K1][K2]        charge grid Q, then potential grid Phi
    DevBuf gridQ;     // float  copy of Q kept for sqeq_pme_grid (diagnostics only when enabled)
    DevBuf spec;      // float2 [K0][K1][K2/2+1]
    DevBuf ew_tab;    // float2 [ntab][n]  per-atom phase tables of the regular-Ewald kernels (ewald.cu)
    DevBuf ew_sf;     // float2 [nk]       structure factors / coefficients
    DevBuf tabs;      // float  per-axis tables: |b|^2, gaussian, mtilde^2  (3 x (K0+K1+K2))

    // ---- per-evaluation atom workspaces (sorted = cell-major order of the list) ----
    DevBuf xq;        // float4 [n]  wrapped x,y,z (build-time image) + charge
    DevBuf frac;      // float4 [n]  fractional offsets w_x,w_y,w_z in [0,1), charge
    DevBuf base;      // int4   [n]  floor grid index f_x,f_y,f_z
    DevBuf real_out;  // float4 [n]  F_real xyz, phi_real   (sorted order)
    DevBuf rec_out;   // float4 [n]  F_rec  xyz, phi_rec    (sorted order)
    DevBuf scal;      // double [16] device scalars (energy sums, dots)
    double* h_scal = nullptr;  // pinned host mirror
    void* h_nl = nullptr;      // pinned scratch of the neighbour build (256 B)
    bool last_had_force = false;
    bool energy_pending = false;   // scal[0] holds the energy of the last enqueued evaluation
    int64_t last_n = 0;

    // ---- Krylov / MD workspaces ----
    DevBuf kry_V;     // double [m+1][n+1]
    DevBuf kry_w;     // double [n+1]
    DevBuf kry_h;     // double [m+2]
    DevBuf vec_f[6];  // float  [n] scratch charge / potential vectors
    DevBuf vec_d[6];  // double [n] scratch
    DevBuf vec_f3[2]; // float  [n][3] scratch forces
    double diag_box[3] = {0, 0, 0}, diag_alpha = 0, diag_val = 0;     // ewald_self_diag of the last (box, alpha)
    // stand-in O-O repulsion (md.cu): the oxygens' list positions, cell by cell, for the list with this serial
    DevBuf rep_oslot, rep_ostart;
    DevBuf qeq_vin;                       // qeq.cu: fixed input buffer of the graph-replayed mat-vec
    DevBuf batch_q, batch_r;              // sqeq_coulomb_fixed_batch: [4][n] sorted charge vectors / real-space potentials
    const void* rep_nl = nullptr;
    uint64_t rep_serial = 0;
    GeomCache gc;
    struct { bool valid = false, tiles = false; int order = 0, nt = 0, K[3] = {0, 0, 0}, nc[3] = {0, 0, 0}; size_t bytes = 0;
             alignas(8) unsigned char blob[128]; } tile_plan;     // cached TileGeom of the PME tile kernels (pme.cu)
    // sqeq_geometry_set / sqeq_coulomb_fixed session
    uint64_t geom_serial = 0;             // counts prep_atoms calls: which positions xq/frac/base hold
    struct { const sqeq_nlist* nl = nullptr; uint64_t serial = 0, geom_serial = 0; int64_t n = 0; double box[3] = {0, 0, 0}; double rc = 0, alpha = 0; } fixed;
    uint64_t nl_serial = 0;               // build counter: tells a list from a later one at the same address
    DevBuf stage[4];  // device staging for sqeq_coulomb_host: pos, q, phi, force
    // sqeq_coulomb_host_submit / _wait: two slots, copies on their own streams beside the evaluation stream
    DevBuf slot_buf[2][5];                // pos, q, phi, force, energy (one double)
    cudaStream_t stream_h2d = nullptr, stream_d2h = nullptr;
    cudaEvent_t slot_in[2] = {nullptr, nullptr}, slot_done[2] = {nullptr, nullptr}, slot_out[2] = {nullptr, nullptr};
    bool slot_busy[2] = {false, false};
    bool slot_energy[2] = {false, false};
    double* h_slot_e = nullptr;           // pinned [2]
    // sqeq_shadow_md_run: ring of lagged drift checks (device words, pinned mirror, one event each)
    unsigned* d_ring = nullptr;
    unsigned* h_ring = nullptr;
    cudaEvent_t ring_ev[4] = {nullptr, nullptr, nullptr, nullptr};

    // ---- timing ----
    bool profiling = false;
    std::vector<TimerRec> pending;
    std::vector<cudaEvent_t> free_events;
    double t_total[SQEQ_T_COUNT] = {0};
    int64_t t_count[SQEQ_T_COUNT] = {0};
    int64_t launches = 0;

    // CUDA graphs of launch-bound sequences (sqeq_coulomb_fixed, the shadow-MD step): slot 0 / 1
    struct GraphSlot { uint64_t key = 0; cudaGraphExec_t exec = nullptr; int64_t nlaunch = 0; uint64_t used = 0; } gslot[2 + 12];
    uint64_t gclock = 0;                  // slots 2..13: plain evaluations of small systems, least recently used replaced
    bool graphs = true;                   // SQEQ_GRAPHS=0 / sqeq_set_option("graphs", 0): always launch kernel by kernel

    // live neighbour lists of this context: sqeq_destroy releases their device storage and detaches them, so a
    // handle freed after its context is only deleted (no use of a dead stream or pool)
    std::vector<sqeq_nlist*> lists;
};

struct sqeq_nlist {
    sqeq_ctx* ctx = nullptr;
    int64_t n = 0;
    double box[3] = {0, 0, 0};
    double cutoff = 0;
    int ncell[3] = {1, 1, 1};
    int64_t n_directed = 0;          // directed pairs (sum of row_len)
    int64_t n_slots = 0;             // list slots in use (fmt 1 pads every row to a multiple of 32)
    int max_row = 0;
    // device arrays
    int*      perm = nullptr;        // [n]   sorted index -> caller index
    int*      cell_of = nullptr;     // [n]   cell id of sorted atom
    int*      cell_start = nullptr;  // [ncells+1]
    char4*    wrapc = nullptr;       // [n]   floor(x/L) per axis at build time (sorted order)
    int64_t*  row_start = nullptr;   // [n]   offset of row s in nbr (rows in no particular order; fmt 1: multiples of 32)
    int*      row_len = nullptr;     // [n]   entries of row s
    float*    pos0 = nullptr;        // [n][3] caller order: the positions the list was built from (drift check)
    longlong2* grp_slice = nullptr;  // [cell groups] (first slot, slots used) of the group's reserved slice of nbr
    void*     nbr = nullptr;         // [>= n_slots] entries: fmt 0: uint32 j (27 bits) | image code << 27;
                                     //                          fmt 1: uint16 local index in the group's neighbourhood
    uint64_t  serial = 0;            // ctx->nl_serial at build time
    int       fmt = 0;
    int       max_pop = 0;           // fmt 1: largest neighbourhood population of a group
    int       lshift = 0;            // fmt 1: entries are local index << lshift (4: byte offsets of float4 slots)
    GroupGeom gg;                    // cell groups (cellgroup.cuh)
};

// ---------------------------------------------------------------------------------------------
int sqeq_fail(sqeq_ctx* ctx, int code, const char* fmt, ...);
// Runs `body` (a sequence of launches on ctx->stream with no synchronisation) through a CUDA graph kept in slot
// `slot`: replayed when `key` is unchanged, re-captured (and the executable graph updated in place) when it is not.
// Falls back to running body() directly when graphs are off, stage timing is on, the stream cannot be captured
// (legacy default stream) or the capture fails (e.g. a workspace had to grow: the next call captures).
int graph_run(sqeq_ctx* ctx, int slot, uint64_t key, const std::function<int()>& body);
static inline uint64_t hash_mix(uint64_t h, uint64_t v) { h ^= v + 0x9e3779b97f4a7c15ull + (h << 6) + (h >> 2); return h; }
int sqeq_reserve(sqeq_ctx* ctx, DevBuf& b, size_t bytes);

#define CUDA_TRY(ctx, expr)                                                              \
    do {                                                                                 \
        cudaError_t _e = (expr);                                                         \
        if (_e != cudaSuccess)                                                           \
            return sqeq_fail((ctx), SQEQ_ECUDA, "%s failed: %s (%s:%d)", #expr,          \
                             cudaGetErrorString(_e), __FILE__, __LINE__);                \
    } while (0)

#define SQEQ_TRY(expr)                  \
    do {                                \
        int _r = (expr);                \
        if (_r != SQEQ_OK) return _r;   \
    } while (0)

#define KERNEL_CHECK(ctx)                                                                \
    do {                                                                                 \
        (ctx)->launches++;                                                               \
        cudaError_t _e = cudaGetLastError();                                             \
        if (_e != cudaSuccess)                                                           \
            return sqeq_fail((ctx), SQEQ_ECUDA, "kernel launch failed: %s (%s:%d)",      \
                             cudaGetErrorString(_e), __FILE__, __LINE__);                \
    } while (0)

// RAII stage timer: records a CUDA-event pair on the given stream when profiling is on.
struct StageTimer {
    sqeq_ctx* ctx;
    cudaStream_t st;
    int idx = -1;
    StageTimer(sqeq_ctx* c, int stage, cudaStream_t s = nullptr);
    ~StageTimer();
};

#ifdef __CUDACC__
// ---- programmatic dependent launch (PTX griddepcontrol; guide: "PDL") --------------------------------------------
// A kernel launched with launch_pdl may start while the kernel before it in the stream is still draining: its
// blocks become resident as that kernel's last blocks retire and run their prologue (index arithmetic, constant
// tables) up to pdl_wait(), which returns when the previous kernel has completed and its writes are visible.  Rules
// kept throughout: pdl_trigger() is the first statement of every kernel that may be followed by such a launch;
// pdl_wait() comes before the first access to anything an earlier kernel wrote or still reads; EVERY kernel launched
// with launch_pdl executes pdl_wait() in all its threads (completion of a kernel then implies completion of all before
// it); and NO non-coherent load (const __restrict__ pointer, __ldg: LDG.CONSTANT) of anything the previous kernel
// wrote -- the block may sit on an SM whose L1 still holds the old lines, and only ordinary loads are made coherent
// by the wait (measured: a const __restrict__ input gave wrong transforms at cfg 2).  Both are no-ops in a kernel
// launched the ordinary way.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <class... KArgs, class... Args>
static inline cudaError_t launch_pdl(sqeq_ctx* ctx, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                     Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    // not beside the persistent real-space grid of the side-stream schedule: blocks that wait for the kernel ahead
    // would hold the one block slot per SM that grid leaves free (measured: 0.525 instead of 0.517 ms per step)
    cfg.numAttrs = (ctx->pdl_off || ctx->overlap_now) ? 0 : 1;
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// Sums four per-lane values over the warp with 6 shuffles instead of 20: the first two butterfly steps
// halve the number of values a lane carries (lanes keep one half of the values and send the other),
// the last three are an ordinary butterfly.  On return lane 0 holds the sum of a, lane 8 of b, lane 16 of
// c and lane 24 of d (in the returned value).
__device__ __forceinline__ float warp_reduce4(float a, float b, float c, float d, int lane)
{
    const bool hi16 = lane & 16, hi8 = lane & 8;
    float k0 = hi16 ? c : a, k1 = hi16 ? d : b;             // keep
    k0 += __shfl_xor_sync(0xffffffffu, hi16 ? a : c, 16);
    k1 += __shfl_xor_sync(0xffffffffu, hi16 ? b : d, 16);
    float k = hi8 ? k1 : k0;
    k += __shfl_xor_sync(0xffffffffu, hi8 ? k0 : k1, 8);
    k += __shfl_xor_sync(0xffffffffu, k, 4);
    k += __shfl_xor_sync(0xffffffffu, k, 2);
    k += __shfl_xor_sync(0xffffffffu, k, 1);
    return k;
}
#endif

static inline int ceil_div(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// ---- stage entry points (implemented in the .cu files) ----
int nl_build_impl(sqeq_ctx* ctx, int64_t n, const float* pos, const double box[3], double cutoff,
                  sqeq_nlist** out);
void nl_release(sqeq_nlist* nl);
void nl_release_storage(sqeq_nlist* nl);
int nl_export_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, int32_t* i, int32_t* j, int8_t* shift3);
int nl_export_rows_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, int mode, int K, int32_t* oi, int32_t* oj, int8_t* shift3,
                        int32_t* counts);
int nl_max_drift_enqueue(sqeq_ctx* ctx, const sqeq_nlist* nl, const float* pos, const float* vel, double dt,
                         unsigned* d_out);
int nl_max_drift_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, const float* pos, const float* vel, double dt,
                      double* max_drift);

// Re-gather positions/charges into the list's order (and PME fractional coordinates if K != null).
int prep_atoms(sqeq_ctx* ctx, const sqeq_nlist* nl, const float* pos, const float* q,
               const int* K, cudaStream_t st);
// Only refresh the charge component (fixed geometry, new Krylov vector). q may be float or double.
int prep_charges(sqeq_ctx* ctx, const sqeq_nlist* nl, const float* q_f, const double* q_d,
                 cudaStream_t st);
int realspace_run(sqeq_ctx* ctx, const sqeq_nlist* nl, double rc, double alpha, bool want_force,
                  cudaStream_t st, int geom = GEOM_NEW, bool want_phi = true);
int realspace_cached_multi(sqeq_ctx* ctx, const sqeq_nlist* nl, int nvec, const float* q, cudaStream_t st);
int realspace_multi_select(sqeq_ctx* ctx, const sqeq_nlist* nl, int v, cudaStream_t st);
int pme_setup(sqeq_ctx* ctx, const double box[3], double alpha, const int grid[3], int order);
// nl supplies the cell-major atom runs the shared-memory tiles are built on (NULL: global kernels)
int pme_run(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3], bool want_force,
            bool want_energy, cudaStream_t st);
// fftx.cu: register-resident two-step version of the fused x-axis pass, for the x extents it is built for
bool xline2_supported(int K0);
int xline2_run(sqeq_ctx* ctx, int K0, int K1, int K2h, int K2, const float* tab, float inv_piV, const float2* W,
               float2* spec, double* e_out, cudaStream_t st);
int yline_run(sqeq_ctx* ctx, int K0, int K1, int K2h, const float2* W, float2* spec, bool inverse, cudaStream_t st);
// fftz.cu: z-axis real-to-complex / complex-to-real passes (layouts as cuFFT's R2C/C2R, unnormalised)
bool zline_supported(int K2);
int zline_run(sqeq_ctx* ctx, int nlines, int K2, const float2* W, float* grid, float2* spec, bool inverse, cudaStream_t st);
int assemble_run(sqeq_ctx* ctx, const sqeq_nlist* nl, double alpha, float* phi, float* force,
                 bool want_energy, bool field_mode, cudaStream_t st);
// Full evaluation on prepared geometry (used by coulomb, qeq and md drivers).
// field_mode: `force` receives the per-unit-charge field f_i (F_i = q_i f_i) instead of F_i.
// geom = GEOM_FIXED: the caller evaluates several charge vectors on the positions of the last prep_atoms; the
// first such evaluation writes the geometry cache, later ones read it (phi may then be NULL: field only).
int coulomb_eval(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3], double rc,
                 double alpha, float* phi, float* force, bool want_energy, bool field_mode = false,
                 int geom = GEOM_NEW);

// Generic restarted/unrestarted GMRES on device fp64 vectors (qeq.cu); x_out points into ctx->kry_w.
int gmres_solve(sqeq_ctx* ctx, int64_t len, const std::function<int(const double*, double*)>& apply,
                const std::function<int(double*)>& load_rhs, double tol, int max_iter, int restart,
                double** x_out, int* iters_out, double* relres_out, bool* converged_out,
                const double* x0 = nullptr, const double* dinv = nullptr);
int qeq_solve_prepared(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3], double rc, double alpha,
                       double ke, const float* chi, const float* J, double total_charge, double tol, int max_iter,
                       int restart, bool jacobi, bool warm, double* q_io, double* lambda_io, int* iters_out,
                       double* relres_out, bool* converged_out);
double ewald_self_diag(const double box[3], double alpha);
int validate_coulomb_args(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3],
                          double rc, double alpha, const int grid[3], int order, const char* who);
