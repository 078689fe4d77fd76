// api.cu -- C-ABI entry points of libsqeq: context, error reporting, argument validation,
// per-stage event timing, and the sqeq_coulomb orchestration (include/sqeq.h).
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>

#include "common.cuh"

static thread_local char g_create_err[512] = "";

int sqeq_fail(sqeq_ctx* ctx, int code, const char* fmt, ...)
{
    char* dst = ctx ? ctx->err : g_create_err;
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(dst, 512, fmt, ap);
    va_end(ap);
    return code;
}

int sqeq_reserve(sqeq_ctx* ctx, DevBuf& b, size_t bytes)
{
    if (bytes <= b.cap) return SQEQ_OK;
    if (b.p) {
        CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
        if (ctx->stream2) CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream2));
        cudaFree(b.p);
        b.p = nullptr;
        b.cap = 0;
    }
    size_t want = bytes + bytes / 8 + 256;
    cudaError_t e = cudaMalloc(&b.p, want);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return sqeq_fail(ctx, SQEQ_ENOMEM, "cudaMalloc(%zu bytes) failed: %s", want,
                         cudaGetErrorString(e));
    }
    b.cap = want;
    return SQEQ_OK;
}

int graph_run(sqeq_ctx* ctx, int slot, uint64_t key, const std::function<int()>& body)
{
    cudaStream_t st = ctx->stream;
    if (!ctx->graphs || ctx->profiling || st == nullptr || st == cudaStreamLegacy) return body();
    if (slot == 2) {
        // a family of slots: the one holding this key, else the least recently used
        int best = 2;
        for (int k = 2; k < 14; ++k) {
            if (ctx->gslot[k].exec && ctx->gslot[k].key == key) { best = k; break; }
            if (ctx->gslot[k].used < ctx->gslot[best].used) best = k;
        }
        slot = best;
    }
    auto& g = ctx->gslot[slot];
    g.used = ++ctx->gclock;
    if (!(g.exec && g.key == key)) {
        const int64_t l0 = ctx->launches;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
            cudaGetLastError();
            return body();
        }
        const int r = body();
        cudaGraph_t graph = nullptr;
        const cudaError_t e = cudaStreamEndCapture(st, &graph);
        const int64_t nl = ctx->launches - l0;
        ctx->launches = l0;
        if (r != SQEQ_OK || e != cudaSuccess || !graph) {
            cudaGetLastError();
            if (graph) cudaGraphDestroy(graph);
            if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
            return body();                      // plain run; it also brings workspaces to size for the next capture
        }
        bool ok = false;
        if (g.exec) {
            cudaGraphExecUpdateResultInfo info;
            ok = cudaGraphExecUpdate(g.exec, graph, &info) == cudaSuccess;
            if (!ok) { cudaGetLastError(); cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
        }
        if (!ok) ok = cudaGraphInstantiate(&g.exec, graph, 0) == cudaSuccess;
        cudaGraphDestroy(graph);
        if (!ok) { cudaGetLastError(); g.exec = nullptr; return body(); }
        g.key = key;
        g.nlaunch = nl;
    }
    CUDA_TRY(ctx, cudaGraphLaunch(g.exec, st));
    ctx->launches += g.nlaunch;
    return SQEQ_OK;
}

StageTimer::StageTimer(sqeq_ctx* c, int stage, cudaStream_t s) : ctx(c), st(s ? s : c->stream)
{
    if (!ctx->profiling) return;
    TimerRec r;
    r.stage = stage;
    for (cudaEvent_t* e : {&r.a, &r.b}) {
        if (!ctx->free_events.empty()) {
            *e = ctx->free_events.back();
            ctx->free_events.pop_back();
        } else {
            cudaEventCreate(e);
        }
    }
    cudaEventRecord(r.a, st);
    idx = (int)ctx->pending.size();
    ctx->pending.push_back(r);
}

StageTimer::~StageTimer()
{
    if (idx >= 0) cudaEventRecord(ctx->pending[idx].b, st);
}

extern "C" {

const char* sqeq_version(void) { return "sqeq-b200 0.1 (sm_100a)"; }

const char* sqeq_last_error(const sqeq_ctx* ctx) { return ctx ? ctx->err : g_create_err; }

int sqeq_create(sqeq_ctx** out, int device, void* cuda_stream)
{
    if (!out) return sqeq_fail(nullptr, SQEQ_EINVAL, "sqeq_create: out is NULL");
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return sqeq_fail(nullptr, SQEQ_ECUDA,
                         "sqeq_create: no CUDA device available (%s); libsqeq has no CPU fallback",
                         e != cudaSuccess ? cudaGetErrorString(e) : "device count 0");
    }
    if (device < 0 || device >= ndev)
        return sqeq_fail(nullptr, SQEQ_EINVAL, "sqeq_create: device %d out of range [0,%d)", device, ndev);
    e = cudaSetDevice(device);
    if (e != cudaSuccess)
        return sqeq_fail(nullptr, SQEQ_ECUDA, "cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
    sqeq_ctx* ctx = new sqeq_ctx();
    ctx->device = device;
    ctx->stream = (cudaStream_t)cuda_stream;
    cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, device);
    e = cudaStreamCreateWithFlags(&ctx->stream2, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_join, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&ctx->h_scal, 16 * sizeof(double));
    if (e == cudaSuccess) e = cudaMallocHost(&ctx->h_nl, 256);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->scal.p, 16 * sizeof(double));
    if (e == cudaSuccess) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = device;
        e = cudaMemPoolCreate(&ctx->pool, &props);
        if (e == cudaSuccess) {
            uint64_t keep = UINT64_MAX;       // never hand memory back to the driver between rebuilds
            e = cudaMemPoolSetAttribute(ctx->pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
    }
    if (e != cudaSuccess) {
        sqeq_fail(nullptr, SQEQ_ECUDA, "sqeq_create: %s", cudaGetErrorString(e));
        delete ctx;
        return SQEQ_ECUDA;
    }
    ctx->scal.cap = 16 * sizeof(double);
    const char* env = getenv("SQEQ_PME_TILES");
    ctx->pme_tiles_off = env && env[0] == '0';
    env = getenv("SQEQ_SPREAD_FLOAT");
    ctx->spread_float = env && env[0] == '1';
    env = getenv("SQEQ_OVERLAP");
    ctx->overlap = env ? atoi(env) : 1;
    env = getenv("SQEQ_REAL_LEAN_BLOCKS");          // persistent real-space blocks per SM beside the side stream
    ctx->real_lean_blocks = env && atoi(env) > 0 ? atoi(env) : 2;
    env = getenv("SQEQ_REAL_STAGED");
    ctx->real_staged_off = env && env[0] == '0';
    env = getenv("SQEQ_PME_ATOM_THREADS");
    ctx->pme_atom_threads = env ? atoi(env) : 1;
    env = getenv("SQEQ_PAIRS_STAGED");
    ctx->pairs_staged_off = env && env[0] == '0';
    env = getenv("SQEQ_REAL_TMA");
    ctx->real_tma = env && env[0] == '1';
    env = getenv("SQEQ_FFT_FUSED");
    ctx->fft_fused_off = env && env[0] == '0';
    env = getenv("SQEQ_PDL");
    ctx->pdl_off = env && env[0] == '0';
    env = getenv("SQEQ_FFT_OWN");
    ctx->fft_own_off = env && env[0] == '0';
    env = getenv("SQEQ_FFT_XLINE2");
    ctx->fft_xline2_off = env && env[0] == '0';
    env = getenv("SQEQ_GRAPHS");
    ctx->graphs = !(env && env[0] == '0');
    *out = ctx;
    return SQEQ_OK;
}

int sqeq_destroy(sqeq_ctx* ctx)
{
    if (!ctx) return SQEQ_OK;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    if (ctx->stream2) cudaStreamSynchronize(ctx->stream2);
    // lists that outlive their context: release the device storage now, leave a detached handle behind
    for (sqeq_nlist* nl : ctx->lists) {
        nl_release_storage(nl);
        nl->ctx = nullptr;
    }
    ctx->lists.clear();
    cudaStreamSynchronize(ctx->stream);
    if (ctx->plans_ok) {
        cufftDestroy(ctx->plan_r2c);
        cufftDestroy(ctx->plan_c2r);
    }
    if (ctx->xf_ok) {
        cufftDestroy(ctx->plan2_r2c);
        cufftDestroy(ctx->plan2_c2r);
    }
    DevBuf* bufs[] = {&ctx->gc.idx, &ctx->gc.t, &ctx->gc.len, &ctx->ew_tab, &ctx->ew_sf, &ctx->xf_tw,
                      &ctx->grid, &ctx->gridQ, &ctx->spec, &ctx->tabs, &ctx->xq, &ctx->frac,
                      &ctx->base, &ctx->real_out, &ctx->rec_out, &ctx->scal, &ctx->kry_V,
                      &ctx->kry_w, &ctx->kry_h, &ctx->rep_oslot, &ctx->rep_ostart, &ctx->batch_q, &ctx->batch_r, &ctx->qeq_vin};
    for (DevBuf* b : bufs)
        if (b->p) cudaFree(b->p);
    for (auto& b : ctx->vec_f) if (b.p) cudaFree(b.p);
    for (auto& b : ctx->vec_d) if (b.p) cudaFree(b.p);
    for (auto& b : ctx->vec_f3) if (b.p) cudaFree(b.p);
    for (auto& b : ctx->stage) if (b.p) cudaFree(b.p);
    if (ctx->h_scal) cudaFreeHost(ctx->h_scal);
    if (ctx->h_nl) cudaFreeHost(ctx->h_nl);
    if (ctx->h_kry) cudaFreeHost(ctx->h_kry);
    for (auto& e : ctx->kry_ev) if (e) cudaEventDestroy(e);
    if (ctx->h_slot_e) cudaFreeHost(ctx->h_slot_e);
    if (ctx->h_ring) cudaFreeHost(ctx->h_ring);
    if (ctx->d_ring) cudaFree(ctx->d_ring);
    for (auto& e : ctx->ring_ev) if (e) cudaEventDestroy(e);
    for (auto& g : ctx->gslot) if (g.exec) cudaGraphExecDestroy(g.exec);
    for (int k = 0; k < 2; ++k) {
        if (ctx->slot_in[k]) cudaEventDestroy(ctx->slot_in[k]);
        if (ctx->slot_done[k]) cudaEventDestroy(ctx->slot_done[k]);
        if (ctx->slot_out[k]) cudaEventDestroy(ctx->slot_out[k]);
        for (int b = 0; b < 5; ++b)
            if (ctx->slot_buf[k][b].p) cudaFree(ctx->slot_buf[k][b].p);
    }
    if (ctx->stream_h2d) cudaStreamDestroy(ctx->stream_h2d);
    if (ctx->stream_d2h) cudaStreamDestroy(ctx->stream_d2h);
    for (auto& r : ctx->pending) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto& e : ctx->free_events) cudaEventDestroy(e);
    if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
    if (ctx->ev_join) cudaEventDestroy(ctx->ev_join);
    if (ctx->stream2) cudaStreamDestroy(ctx->stream2);
    if (ctx->pool) cudaMemPoolDestroy(ctx->pool);
    delete ctx;
    return SQEQ_OK;
}

// ---------------------------------------------------------------------------- profiling
static int drain_timers(sqeq_ctx* ctx)
{
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream2));
    for (auto& r : ctx->pending) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) {
            ctx->t_total[r.stage] += ms;
            ctx->t_count[r.stage] += 1;
        } else {
            cudaGetLastError();
        }
        ctx->free_events.push_back(r.a);
        ctx->free_events.push_back(r.b);
    }
    ctx->pending.clear();
    return SQEQ_OK;
}

int sqeq_profile_enable(sqeq_ctx* ctx, int on)
{
    if (!ctx) return SQEQ_EINVAL;
    SQEQ_TRY(drain_timers(ctx));
    ctx->profiling = on != 0;
    return SQEQ_OK;
}

int sqeq_profile_reset(sqeq_ctx* ctx)
{
    if (!ctx) return SQEQ_EINVAL;
    SQEQ_TRY(drain_timers(ctx));
    for (int s = 0; s < SQEQ_T_COUNT; ++s) { ctx->t_total[s] = 0; ctx->t_count[s] = 0; }
    return SQEQ_OK;
}

int sqeq_profile_read(sqeq_ctx* ctx, int stage, double* total_ms, int64_t* launches)
{
    if (!ctx || stage < 0 || stage >= SQEQ_T_COUNT)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_profile_read: bad stage %d", stage);
    SQEQ_TRY(drain_timers(ctx));
    if (total_ms) *total_ms = ctx->t_total[stage];
    if (launches) *launches = ctx->t_count[stage];
    return SQEQ_OK;
}

int sqeq_set_option(sqeq_ctx* ctx, const char* name, int value)
{
    if (!ctx || !name) return SQEQ_EINVAL;
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    if (!strcmp(name, "graphs")) ctx->graphs = value != 0;
    else if (!strcmp(name, "overlap")) ctx->overlap = value;
    else if (!strcmp(name, "fft_fused")) ctx->fft_fused_off = value == 0;
    else if (!strcmp(name, "pdl")) ctx->pdl_off = value == 0;
    else if (!strcmp(name, "fft_own")) ctx->fft_own_off = value == 0;
    else if (!strcmp(name, "fft_xline2")) ctx->fft_xline2_off = value == 0;
    else if (!strcmp(name, "real_tma")) ctx->real_tma = value != 0;
    else if (!strcmp(name, "pairs_staged")) ctx->pairs_staged_off = value == 0;
    else if (!strcmp(name, "pme_atom_threads")) ctx->pme_atom_threads = value;
    else if (!strcmp(name, "pme_atom_sched")) ctx->pme_atom_sched = value;
    else if (!strcmp(name, "pme_tiles")) { ctx->pme_tiles_off = value == 0; ctx->tile_plan.valid = false; }
    else if (!strcmp(name, "spread_float")) { ctx->spread_float = value != 0; ctx->tile_plan.valid = false; }
    else if (!strcmp(name, "real_staged")) ctx->real_staged_off = value == 0;
    else if (!strcmp(name, "real_lean_blocks")) { if (value < 1) return sqeq_fail(ctx, SQEQ_EINVAL, "real_lean_blocks must be >= 1"); ctx->real_lean_blocks = value; }
    else return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_set_option: unknown option '%s'", name);
    for (auto& g : ctx->gslot) if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
    return SQEQ_OK;
}

int sqeq_launch_count(sqeq_ctx* ctx, int64_t* launches, int reset)
{
    if (!ctx) return SQEQ_EINVAL;
    if (launches) *launches = ctx->launches;
    if (reset) ctx->launches = 0;
    return SQEQ_OK;
}

// ---------------------------------------------------------------------------- neighbour list
static int check_box(sqeq_ctx* ctx, const double box[3], const char* who)
{
    if (!box) return sqeq_fail(ctx, SQEQ_EINVAL, "%s: box is NULL", who);
    for (int d = 0; d < 3; ++d)
        if (!(box[d] > 0.0) || !isfinite(box[d]))
            return sqeq_fail(ctx, SQEQ_EINVAL, "%s: box[%d] = %g must be finite and > 0", who, d, box[d]);
    return SQEQ_OK;
}

int sqeq_nl_build(sqeq_ctx* ctx, int64_t n, const float* pos, const double box[3], double cutoff,
                  sqeq_nlist** out)
{
    if (!ctx) return SQEQ_EINVAL;
    if (!out) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_build: out is NULL");
    *out = nullptr;
    if (n <= 0 || n >= (1LL << 27))
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_build: n = %lld must be in [1, 2^27)", (long long)n);
    if (!pos) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_build: pos is NULL");
    SQEQ_TRY(check_box(ctx, box, "sqeq_nl_build"));
    double lmin = fmin(box[0], fmin(box[1], box[2]));
    if (!(cutoff > 0.0) || !isfinite(cutoff) || !(cutoff < 0.5 * lmin))
        return sqeq_fail(ctx, SQEQ_EINVAL,
                         "sqeq_nl_build: cutoff %g must satisfy 0 < cutoff < min(box)/2 = %g "
                         "(minimum image needs box > 2*cutoff)", cutoff, 0.5 * lmin);
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return nl_build_impl(ctx, n, pos, box, cutoff, out);
}

int sqeq_nl_count(const sqeq_nlist* nl, int64_t* n_pairs_unique)
{
    if (!nl || !n_pairs_unique) return SQEQ_EINVAL;
    *n_pairs_unique = nl->n_directed / 2;
    return SQEQ_OK;
}

int sqeq_nl_info(const sqeq_nlist* nl, int ncell[3], int64_t* n_directed, int* max_row)
{
    if (!nl) return SQEQ_EINVAL;
    if (ncell) for (int d = 0; d < 3; ++d) ncell[d] = nl->ncell[d];
    if (n_directed) *n_directed = nl->n_directed;
    if (max_row) *max_row = nl->max_row;
    return SQEQ_OK;
}

int sqeq_nl_export(sqeq_ctx* ctx, const sqeq_nlist* nl, int32_t* i, int32_t* j, int8_t* shift3)
{
    if (!ctx) return SQEQ_EINVAL;
    if (!nl || nl->ctx != ctx) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_export: list does not belong to this context");
    if (nl->n_directed > 0 && (!i || !j || !shift3))
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_export: NULL output");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return nl_export_impl(ctx, nl, i, j, shift3);
}

int sqeq_nl_export_ellpack(sqeq_ctx* ctx, const sqeq_nlist* nl, int K, int32_t* nbr, int8_t* shift3, int32_t* counts)
{
    if (!ctx) return SQEQ_EINVAL;
    if (!nl || nl->ctx != ctx) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_export_ellpack: list does not belong to this context");
    if (!nbr || !shift3 || K < 1) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_export_ellpack: NULL output or K < 1");
    if (K < nl->max_row)
        return sqeq_fail(ctx, SQEQ_ECAPACITY, "sqeq_nl_export_ellpack: K = %d but the longest row has %d neighbours", K, nl->max_row);
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return nl_export_rows_impl(ctx, nl, 0, K, nullptr, nbr, shift3, counts);
}

int sqeq_nl_export_coo(sqeq_ctx* ctx, const sqeq_nlist* nl, int32_t* i, int32_t* j, int8_t* shift3)
{
    if (!ctx) return SQEQ_EINVAL;
    if (!nl || nl->ctx != ctx) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_export_coo: list does not belong to this context");
    if (nl->n_directed > 0 && (!i || !j || !shift3)) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_export_coo: NULL output");
    if (nl->n_directed == 0) return SQEQ_OK;
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return nl_export_rows_impl(ctx, nl, 1, 0, i, j, shift3, nullptr);
}

int sqeq_nl_entry_bytes(const sqeq_nlist* nl, int* bytes)
{
    if (!nl || !bytes) return SQEQ_EINVAL;
    *bytes = nl->fmt == 1 ? 2 : 4;
    return SQEQ_OK;
}

int sqeq_nl_layout(const sqeq_nlist* nl, int64_t* n_slots, int* entry_shift, int* max_neighbourhood)
{
    if (!nl) return SQEQ_EINVAL;
    if (n_slots) *n_slots = nl->n_slots;
    if (entry_shift) *entry_shift = nl->lshift;
    if (max_neighbourhood) *max_neighbourhood = nl->max_pop;
    return SQEQ_OK;
}

int sqeq_nl_max_drift(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, double* max_drift)
{
    if (!ctx) return SQEQ_EINVAL;
    if (!nl || nl->ctx != ctx || n != nl->n || !pos || !max_drift)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_max_drift: list/context/n mismatch or NULL argument");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return nl_max_drift_impl(ctx, nl, pos, nullptr, 0.0, max_drift);
}

int sqeq_nl_max_drift_ahead(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const float* vel,
                            double dt, double* max_drift)
{
    if (!ctx) return SQEQ_EINVAL;
    if (!nl || nl->ctx != ctx || n != nl->n || !pos || !vel || !max_drift)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_nl_max_drift_ahead: list/context/n mismatch or NULL argument");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    return nl_max_drift_impl(ctx, nl, pos, vel, dt, max_drift);
}

int sqeq_nl_free(sqeq_nlist* nl)
{
    if (!nl) return SQEQ_OK;
    if (!nl->ctx) { delete nl; return SQEQ_OK; }
    cudaSetDevice(nl->ctx->device);
    nl_release(nl);      // stream-ordered frees into the context's pool: no synchronisation
    return SQEQ_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------- coulomb
int validate_coulomb_args(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3],
                          double rc, double alpha, const int grid[3], int order, const char* who)
{
    if (!nl || nl->ctx != ctx)
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: neighbour list missing or from another context", who);
    if (n != nl->n)
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: n = %lld but the list was built for %lld atoms", who,
                         (long long)n, (long long)nl->n);
    SQEQ_TRY(check_box(ctx, box, who));
    for (int d = 0; d < 3; ++d)
        if (box[d] != nl->box[d])
            return sqeq_fail(ctx, SQEQ_EINVAL, "%s: box differs from the box the list was built with", who);
    if (!(rc > 0.0) || !(rc <= nl->cutoff))
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: rc = %g must satisfy 0 < rc <= list cutoff %g", who, rc, nl->cutoff);
    if (!(alpha > 0.0) || !isfinite(alpha))
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: alpha = %g must be > 0", who, alpha);
    if (order < 4 || order > 8)
        return sqeq_fail(ctx, SQEQ_EINVAL, "%s: spline order %d unsupported (4 to 8)", who, order);
    if (!grid) return sqeq_fail(ctx, SQEQ_EINVAL, "%s: grid is NULL", who);
    for (int d = 0; d < 3; ++d)
        if (grid[d] < order || grid[d] > 2048 || (grid[d] & 1))
            return sqeq_fail(ctx, SQEQ_EINVAL, "%s: grid[%d] = %d must be even and in [order, 2048]", who, d, grid[d]);
    return SQEQ_OK;
}

int coulomb_eval(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const double box[3], double rc,
                 double alpha, float* phi, float* force, bool want_energy, bool field_mode, int geom)
{
    const bool want_force = force != nullptr;
    const bool want_phi = phi != nullptr || want_energy;
    // One stream by default.  SQEQ_OVERLAP=1 runs the real-space sum as a persistent grid of two lean
    // (32-register) blocks per SM and forks PME onto the side stream, where one PME block per SM fits beside
    // them: at cfg 4 the device-side step goes from 0.624 to 0.587 ms, but a single synchronous evaluation
    // (sqeq_coulomb_host) gets slower (0.94 -> 1.02 ms), so it stays an option.  Never
    // with stage timing on, where every event pair brackets one kernel running alone.
    // Potential-only evaluations are excluded from the automatic choice: their real-space kernel is list-bandwidth
    // bound and loses more as two persistent blocks per SM than the overlap returns (cfg 4: 0.472 ms against 0.398).
    const bool overlap = !ctx->profiling && geom == GEOM_NEW && nl->fmt == 1 &&
                         (ctx->overlap >= 2 || (ctx->overlap == 1 && ctx->throughput_call && want_force));
    ctx->overlap_now = overlap;
    if (!overlap) {
        SQEQ_TRY(pme_run(ctx, nl, n, box, want_force, false, ctx->stream));
        SQEQ_TRY(realspace_run(ctx, nl, rc, alpha, want_force, ctx->stream, geom, want_phi));
    } else {
        CUDA_TRY(ctx, cudaEventRecord(ctx->ev_fork, ctx->stream));
        CUDA_TRY(ctx, cudaStreamWaitEvent(ctx->stream2, ctx->ev_fork, 0));
        SQEQ_TRY(realspace_run(ctx, nl, rc, alpha, want_force, ctx->stream));     // first: its persistent blocks settle
        SQEQ_TRY(pme_run(ctx, nl, n, box, want_force, false, ctx->stream2));
        CUDA_TRY(ctx, cudaEventRecord(ctx->ev_join, ctx->stream2));
        CUDA_TRY(ctx, cudaStreamWaitEvent(ctx->stream, ctx->ev_join, 0));
    }
    SQEQ_TRY(assemble_run(ctx, nl, alpha, phi, force, want_energy, field_mode, ctx->stream));
    ctx->last_had_force = want_force;
    ctx->last_n = n;
    return SQEQ_OK;
}

static int coulomb_enqueue_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                                const float* q, const double box[3], double rc, double alpha,
                                const int grid[3], int order, float* phi, float* force, int want_energy, bool throughput);

extern "C" int sqeq_coulomb_enqueue(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                                    const float* q, const double box[3], double rc, double alpha,
                                    const int grid[3], int order, float* phi, float* force, int want_energy)
{
    return coulomb_enqueue_impl(ctx, nl, n, pos, q, box, rc, alpha, grid, order, phi, force, want_energy, true);
}

// throughput: the caller does not wait for this evaluation (enqueue / pipelined entries): PME may run on the side
// stream beside a persistent real-space grid ("overlap" = 1).  A caller that waits (energy returned, host buffers)
// gets the one-stream schedule, which finishes a single evaluation sooner.
static int coulomb_enqueue_impl(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos,
                                const float* q, const double box[3], double rc, double alpha,
                                const int grid[3], int order, float* phi, float* force, int want_energy, bool throughput)
{
    if (!ctx) return SQEQ_EINVAL;
    ctx->throughput_call = throughput;
    SQEQ_TRY(validate_coulomb_args(ctx, nl, n, box, rc, alpha, grid, order, "sqeq_coulomb"));
    if (!pos || !q) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb: pos or q is NULL");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    SQEQ_TRY(pme_setup(ctx, box, alpha, grid, order));
    auto body = [&]() -> int {
        SQEQ_TRY(prep_atoms(ctx, nl, pos, q, ctx->K, ctx->stream));
        return coulomb_eval(ctx, nl, n, box, rc, alpha, phi, force, want_energy != 0);
    };
    if (n <= 65536) {
        // launch-latency regime (a dozen kernels of a few microseconds each): the evaluation of the same arrays on the
        // same list is one CUDA graph, replayed while the caller updates the arrays in place
        uint64_t key = hash_mix(0x77, nl->serial);
        for (uint64_t v : {(uint64_t)(uintptr_t)pos, (uint64_t)(uintptr_t)q, (uint64_t)(uintptr_t)phi, (uint64_t)(uintptr_t)force,
                           (uint64_t)(want_energy != 0), (uint64_t)throughput, (uint64_t)(ctx->gridQ.p != nullptr), (uint64_t)order, (uint64_t)grid[0], (uint64_t)grid[1],
                           (uint64_t)grid[2]})
            key = hash_mix(key, v);
        double dv[2] = {rc, alpha};
        for (double d : dv) { uint64_t b; memcpy(&b, &d, 8); key = hash_mix(key, b); }
        SQEQ_TRY(graph_run(ctx, 2, key, body));
        ctx->gc.valid = false;              // a replay re-gathers positions without passing through prep_atoms on the host
        ctx->geom_serial++;
        ctx->last_had_force = force != nullptr;
        ctx->last_n = n;
    } else {
        SQEQ_TRY(body());
    }
    ctx->energy_pending = want_energy != 0;
    return SQEQ_OK;
}

extern "C" int sqeq_geometry_set(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const double box[3],
                                 double rc, double alpha, const int grid[3], int order)
{
    if (!ctx) return SQEQ_EINVAL;
    ctx->fixed.nl = nullptr;
    SQEQ_TRY(validate_coulomb_args(ctx, nl, n, box, rc, alpha, grid, order, "sqeq_geometry_set"));
    if (!pos) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_geometry_set: pos is NULL");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    SQEQ_TRY(pme_setup(ctx, box, alpha, grid, order));
    SQEQ_TRY(prep_atoms(ctx, nl, pos, nullptr, ctx->K, ctx->stream));      // charges come with each evaluation
    ctx->fixed.nl = nl; ctx->fixed.serial = nl->serial; ctx->fixed.n = n;
    ctx->fixed.geom_serial = ctx->geom_serial;
    for (int d = 0; d < 3; ++d) ctx->fixed.box[d] = box[d];
    ctx->fixed.rc = rc; ctx->fixed.alpha = alpha;
    return SQEQ_OK;
}

extern "C" int sqeq_coulomb_fixed(sqeq_ctx* ctx, int64_t n, const float* q, float* phi, float* force, int want_energy)
{
    if (!ctx) return SQEQ_EINVAL;
    const sqeq_nlist* nl = ctx->fixed.nl;
    bool alive = false;
    for (const sqeq_nlist* l : ctx->lists) alive = alive || (l == nl && l->serial == ctx->fixed.serial);
    if (!nl || !alive || ctx->geom_serial != ctx->fixed.geom_serial)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_fixed: no geometry set (sqeq_geometry_set), its list was freed, or "
                                           "another evaluation has replaced it");
    if (n != ctx->fixed.n || !q || (!phi && !force))
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_fixed: n differs from the geometry, q is NULL, or no output asked for");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    auto body = [&]() -> int {
        SQEQ_TRY(prep_charges(ctx, nl, q, nullptr, ctx->stream));
        return coulomb_eval(ctx, nl, n, ctx->fixed.box, ctx->fixed.rc, ctx->fixed.alpha, phi, force, want_energy != 0, false,
                            GEOM_FIXED);
    };
    // once the geometry cache exists every evaluation is the same sequence of launches: replay it as a CUDA graph
    // (the launch-latency regime of small systems: 648 atoms are ~12 kernels of a few microseconds each)
    const bool warm = ctx->gc.valid && ctx->gc.nl == nl && ctx->gc.serial == nl->serial && nl->fmt == 1;
    if (warm) {
        uint64_t key = hash_mix(0x51, ctx->geom_serial);
        for (uint64_t v : {(uint64_t)(uintptr_t)q, (uint64_t)(uintptr_t)phi, (uint64_t)(uintptr_t)force, (uint64_t)(want_energy != 0)})
            key = hash_mix(key, v);
        SQEQ_TRY(graph_run(ctx, 0, key, body));
    } else {
        SQEQ_TRY(body());
    }
    ctx->energy_pending = want_energy != 0;
    return SQEQ_OK;
}

// NEXT-1, the batched half: potentials of nvec charge vectors on the fixed geometry.  The real-space part of up to four
// vectors is ONE pass over the geometry cache (its 6 B per entry stream is what bounds the single-vector kernel); the
// reciprocal part runs per vector on the shared prepared geometry (spreading and gathering are bound by their 216
// shared-memory atomics / loads per atom AND vector, the transforms by their points per vector: nothing there is shared
// between vectors but the spline weights).
extern "C" int sqeq_coulomb_fixed_batch(sqeq_ctx* ctx, int64_t n, int nvec, const float* q, float* phi)
{
    if (!ctx) return SQEQ_EINVAL;
    const sqeq_nlist* nl = ctx->fixed.nl;
    bool alive = false;
    for (const sqeq_nlist* l : ctx->lists) alive = alive || (l == nl && l->serial == ctx->fixed.serial);
    if (!nl || !alive || ctx->geom_serial != ctx->fixed.geom_serial)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_fixed_batch: no geometry set (sqeq_geometry_set), its list was freed, or "
                                           "another evaluation has replaced it");
    if (n != ctx->fixed.n || !q || !phi || nvec < 1 || nvec > 64)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_fixed_batch: n differs from the geometry, NULL argument, or nvec outside [1, 64]");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    auto single = [&](int v) -> int {
        SQEQ_TRY(prep_charges(ctx, nl, q + (int64_t)v * n, nullptr, st));
        return coulomb_eval(ctx, nl, n, ctx->fixed.box, ctx->fixed.rc, ctx->fixed.alpha, phi + (int64_t)v * n, nullptr, false, false,
                            GEOM_FIXED);
    };
    int v0 = 0;
    auto warm = [&]() { return ctx->gc.valid && ctx->gc.nl == nl && ctx->gc.serial == nl->serial && ctx->gc.rc == ctx->fixed.rc &&
                               ctx->gc.alpha == ctx->fixed.alpha && nl->fmt == 1; };
    if (!warm()) SQEQ_TRY(single(v0++));                   // the first evaluation on a geometry writes the cache
    auto rest = [&]() -> int {
        int v = v0;
        while (v < nvec) {
            const int nb = nvec - v < 4 ? nvec - v : 4;
            if (nb == 1 || !warm()) {
                SQEQ_TRY(single(v++));
                continue;
            }
            SQEQ_TRY(realspace_cached_multi(ctx, nl, nb, q + (int64_t)v * n, st));
            for (int k = 0; k < nb; ++k) {
                SQEQ_TRY(prep_charges(ctx, nl, q + (int64_t)(v + k) * n, nullptr, st));
                ctx->overlap_now = false;
                SQEQ_TRY(pme_run(ctx, nl, n, ctx->fixed.box, false, false, st));
                SQEQ_TRY(realspace_multi_select(ctx, nl, k, st));
                SQEQ_TRY(assemble_run(ctx, nl, ctx->fixed.alpha, phi + (int64_t)(v + k) * n, nullptr, false, false, st));
            }
            v += nb;
        }
        return SQEQ_OK;
    };
    if (v0 < nvec) {
        if (warm()) {
            // the same sequence of launches every time: replayed as a CUDA graph (as sqeq_coulomb_fixed does)
            uint64_t key = hash_mix(0x52, ctx->geom_serial);
            for (uint64_t x : {(uint64_t)(uintptr_t)q, (uint64_t)(uintptr_t)phi, (uint64_t)nvec, (uint64_t)v0}) key = hash_mix(key, x);
            SQEQ_TRY(graph_run(ctx, 2, key, rest));
        } else {
            SQEQ_TRY(rest());
        }
    }
    ctx->last_had_force = false;
    ctx->last_n = n;
    ctx->energy_pending = false;
    return SQEQ_OK;
}

extern "C" int sqeq_energy_fetch(sqeq_ctx* ctx, double* energy)
{
    if (!ctx || !energy) return SQEQ_EINVAL;
    if (!ctx->energy_pending)
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_energy_fetch: the last evaluation did not reduce an energy");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->scal.p, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    *energy = ctx->h_scal[0];
    return SQEQ_OK;
}

extern "C" int sqeq_coulomb(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos, const float* q,
                 const double box[3], double rc, double alpha, const int grid[3], int order,
                 float* phi, float* force, double* energy)
{
    SQEQ_TRY(coulomb_enqueue_impl(ctx, nl, n, pos, q, box, rc, alpha, grid, order, phi, force, energy != nullptr, energy == nullptr));
    if (energy) SQEQ_TRY(sqeq_energy_fetch(ctx, energy));
    return SQEQ_OK;
}

extern "C" int sqeq_coulomb_host(sqeq_ctx* ctx, const sqeq_nlist* nl, int64_t n, const float* pos_host,
                                 const float* q_host, const double box[3], double rc, double alpha,
                                 const int grid[3], int order, float* phi_host, float* force_host,
                                 double* energy)
{
    if (!ctx) return SQEQ_EINVAL;
    SQEQ_TRY(validate_coulomb_args(ctx, nl, n, box, rc, alpha, grid, order, "sqeq_coulomb_host"));
    if (!pos_host || !q_host) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_host: pos or q is NULL");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->stage[0], sizeof(float) * 3 * n));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->stage[1], sizeof(float) * n));
    SQEQ_TRY(sqeq_reserve(ctx, ctx->stage[2], sizeof(float) * n));
    if (force_host) SQEQ_TRY(sqeq_reserve(ctx, ctx->stage[3], sizeof(float) * 3 * n));
    float* d_pos = (float*)ctx->stage[0].p;
    float* d_q = (float*)ctx->stage[1].p;
    float* d_phi = (float*)ctx->stage[2].p;
    float* d_f = force_host ? (float*)ctx->stage[3].p : nullptr;
    cudaStream_t st = ctx->stream;
    CUDA_TRY(ctx, cudaMemcpyAsync(d_pos, pos_host, sizeof(float) * 3 * n, cudaMemcpyHostToDevice, st));
    CUDA_TRY(ctx, cudaMemcpyAsync(d_q, q_host, sizeof(float) * n, cudaMemcpyHostToDevice, st));
    SQEQ_TRY(pme_setup(ctx, box, alpha, grid, order));
    SQEQ_TRY(prep_atoms(ctx, nl, d_pos, d_q, ctx->K, st));
    ctx->throughput_call = false;
    SQEQ_TRY(coulomb_eval(ctx, nl, n, box, rc, alpha, d_phi, d_f, energy != nullptr));
    if (phi_host) CUDA_TRY(ctx, cudaMemcpyAsync(phi_host, d_phi, sizeof(float) * n, cudaMemcpyDeviceToHost, st));
    if (force_host) CUDA_TRY(ctx, cudaMemcpyAsync(force_host, d_f, sizeof(float) * 3 * n, cudaMemcpyDeviceToHost, st));
    if (energy) CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->scal.p, sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(ctx, cudaStreamSynchronize(st));
    if (energy) *energy = ctx->h_scal[0];
    return SQEQ_OK;
}

// Pipelined form of sqeq_coulomb_host for independent evaluations: the inputs of evaluation k+1 travel to the
// device (copy stream) and the results of evaluation k-1 travel back (second copy stream) while evaluation k
// runs on the context's stream.  Two slots; a slot is free again after sqeq_coulomb_host_wait on it.
static int slot_setup(sqeq_ctx* ctx)
{
    if (ctx->stream_h2d) return SQEQ_OK;
    CUDA_TRY(ctx, cudaStreamCreateWithFlags(&ctx->stream_h2d, cudaStreamNonBlocking));
    CUDA_TRY(ctx, cudaStreamCreateWithFlags(&ctx->stream_d2h, cudaStreamNonBlocking));
    for (int k = 0; k < 2; ++k) {
        CUDA_TRY(ctx, cudaEventCreateWithFlags(&ctx->slot_in[k], cudaEventDisableTiming));
        CUDA_TRY(ctx, cudaEventCreateWithFlags(&ctx->slot_done[k], cudaEventDisableTiming));
        CUDA_TRY(ctx, cudaEventCreateWithFlags(&ctx->slot_out[k], cudaEventDisableTiming));
    }
    CUDA_TRY(ctx, cudaMallocHost((void**)&ctx->h_slot_e, 2 * sizeof(double)));
    return SQEQ_OK;
}

extern "C" int sqeq_coulomb_host_submit(sqeq_ctx* ctx, int slot, const sqeq_nlist* nl, int64_t n,
                                        const float* pos_host, const float* q_host, const double box[3],
                                        double rc, double alpha, const int grid[3], int order,
                                        float* phi_host, float* force_host, int want_energy)
{
    if (!ctx) return SQEQ_EINVAL;
    if (slot < 0 || slot > 1) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_host_submit: slot must be 0 or 1");
    if (ctx->slot_busy[slot])
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_host_submit: slot %d is in flight (call sqeq_coulomb_host_wait)", slot);
    SQEQ_TRY(validate_coulomb_args(ctx, nl, n, box, rc, alpha, grid, order, "sqeq_coulomb_host_submit"));
    if (!pos_host || !q_host) return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_host_submit: pos or q is NULL");
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    SQEQ_TRY(slot_setup(ctx));
    DevBuf* b = ctx->slot_buf[slot];
    const size_t want[5] = {sizeof(float) * 3 * (size_t)n, sizeof(float) * (size_t)n, sizeof(float) * (size_t)n,
                            force_host ? sizeof(float) * 3 * (size_t)n : 0, sizeof(double)};
    for (int k = 0; k < 5; ++k)
        if (want[k] > b[k].cap) {
            // the slot is idle (its last evaluation was waited for), so its buffers can be replaced right away
            if (b[k].p) CUDA_TRY(ctx, cudaFree(b[k].p));
            b[k].p = nullptr;
            b[k].cap = 0;
            CUDA_TRY(ctx, cudaMalloc(&b[k].p, want[k]));
            b[k].cap = want[k];
        }
    float* d_pos = (float*)b[0].p;
    float* d_q = (float*)b[1].p;
    float* d_phi = (float*)b[2].p;
    float* d_f = force_host ? (float*)b[3].p : nullptr;
    CUDA_TRY(ctx, cudaMemcpyAsync(d_pos, pos_host, want[0], cudaMemcpyHostToDevice, ctx->stream_h2d));
    CUDA_TRY(ctx, cudaMemcpyAsync(d_q, q_host, want[1], cudaMemcpyHostToDevice, ctx->stream_h2d));
    CUDA_TRY(ctx, cudaEventRecord(ctx->slot_in[slot], ctx->stream_h2d));
    cudaStream_t st = ctx->stream;
    CUDA_TRY(ctx, cudaStreamWaitEvent(st, ctx->slot_in[slot], 0));
    SQEQ_TRY(pme_setup(ctx, box, alpha, grid, order));
    SQEQ_TRY(prep_atoms(ctx, nl, d_pos, d_q, ctx->K, st));
    ctx->throughput_call = true;
    SQEQ_TRY(coulomb_eval(ctx, nl, n, box, rc, alpha, d_phi, d_f, want_energy != 0));
    if (want_energy)
        CUDA_TRY(ctx, cudaMemcpyAsync(b[4].p, ctx->scal.p, sizeof(double), cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(ctx, cudaEventRecord(ctx->slot_done[slot], st));
    CUDA_TRY(ctx, cudaStreamWaitEvent(ctx->stream_d2h, ctx->slot_done[slot], 0));
    if (phi_host) CUDA_TRY(ctx, cudaMemcpyAsync(phi_host, d_phi, want[2], cudaMemcpyDeviceToHost, ctx->stream_d2h));
    if (force_host) CUDA_TRY(ctx, cudaMemcpyAsync(force_host, d_f, want[3], cudaMemcpyDeviceToHost, ctx->stream_d2h));
    if (want_energy)
        CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_slot_e + slot, b[4].p, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream_d2h));
    CUDA_TRY(ctx, cudaEventRecord(ctx->slot_out[slot], ctx->stream_d2h));
    ctx->slot_busy[slot] = true;
    ctx->slot_energy[slot] = want_energy != 0;
    return SQEQ_OK;
}

extern "C" int sqeq_coulomb_host_wait(sqeq_ctx* ctx, int slot, double* energy)
{
    if (!ctx) return SQEQ_EINVAL;
    if (slot < 0 || slot > 1 || !ctx->slot_busy[slot])
        return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_host_wait: nothing submitted on slot %d", slot);
    CUDA_TRY(ctx, cudaSetDevice(ctx->device));
    CUDA_TRY(ctx, cudaEventSynchronize(ctx->slot_out[slot]));
    ctx->slot_busy[slot] = false;
    if (energy) {
        if (!ctx->slot_energy[slot])
            return sqeq_fail(ctx, SQEQ_EINVAL, "sqeq_coulomb_host_wait: slot %d was submitted without the energy", slot);
        *energy = ctx->h_slot_e[slot];
    }
    return SQEQ_OK;
}
