// api_solve.cu -- C ABI (include/tsm.h): the solver driver (H3, H4, H6, H7), the loop
// accumulators (H8-H10) and the whole-configuration TSM driver (Eq. 2.4).
#include <cmath>
#include <cstdlib>
#include <cstring>

#include <nvtx3/nvToolsExt.h>   // header-only: ranges for an nsys / ncu timeline, no-ops without a profiler attached

#include "tsm_internal.cuh"

namespace {

// NVTX range for one phase of the path (noise / prepare / CG / reconstruct / contract): closes when it goes out of scope
struct Phase {
    explicit Phase(const char* name) { nvtxRangePushA(name); }
    ~Phase() { nvtxRangePop(); }
};

struct Twists {
    TwistCoef zero, one, R, Rinv, Rb, Rbinv, mk2, k, kRinv;
};

Twists make_twists(const tsm_ctx* ctx)
{
    const double k = ctx->kappa, a = 2.0 * ctx->kappa * ctx->mu, n = 1.0 / (1.0 + a * a);
    Twists t;
    t.zero = {0, 0, 0, 0};
    t.one = {1, 0, 1, 0};
    t.R = {1, a, 1, -a};                 // 1 + i a gamma5
    t.Rinv = {n, -a * n, n, a * n};      // (1 - i a gamma5)/(1 + a^2)
    t.Rb = {1, -a, 1, a};                // R(-mu)
    t.Rbinv = {n, a * n, n, -a * n};
    t.mk2 = {-k * k, 0, -k * k, 0};
    t.k = {k, 0, k, 0};
    t.kRinv = {k * n, -k * a * n, k * n, k * a * n};
    return t;
}

// One CG iteration on Mhat^dag Mhat (O5): four stencil launches, two one-block-per-source reductions and
// one fused BLAS launch.  Re<p,q> = <p, Mhat^dag Mhat p> is taken as |Mhat p|^2 = |w|^2 from the epilogue of
// the second stencil launch (same number up to rounding; saves re-reading p and q).  q = Mhat^dag w is never
// stored: the fourth stencil launch applies r -= alpha q in its epilogue and leaves |r|^2 per tile.
int cg_iteration(tsm_ctx* ctx, int prec, int nrhs, const Twists& tw, void* x, void* r, void* p, void* w, void* t, double tol,
                 unsigned long long loop = 0, int in_loop = 0)
{
    int rc;
    if ((rc = launch_dslash(ctx, prec, 1, false, nrhs, p, nullptr, t, {tw.zero, tw.Rinv}, 2))) return rc;   // t = R^-1 D_oe p
    if ((rc = launch_dslash(ctx, prec, 0, false, nrhs, t, p, w, {tw.R, tw.mk2}, 3))) return rc;             // w = Mhat p; |w|^2 per tile
    if ((rc = launch_cg_reduce(ctx, 0, nrhs))) return rc;                                                   // alpha
    if ((rc = launch_dslash(ctx, prec, 1, true, nrhs, w, nullptr, t, {tw.zero, tw.Rbinv}, 2))) return rc;   // t = Rb^-1 D_oe^dag w
    if ((rc = launch_dslash(ctx, prec, 0, true, nrhs, t, w, r, {tw.Rb, tw.mk2}, 6))) return rc;             // r -= alpha Mhat^dag w; |r|^2 per tile
    if ((rc = launch_cg_reduce(ctx, 1, nrhs))) return rc;                                                   // rr'
    return launch_cg_update_xp(ctx, prec, nrhs, x, p, r, tol, loop, in_loop);                               // x += alpha p; p = r + beta p
}

// `iters` CG iterations as ONE CUDA graph launch (captured once per argument set and cached): on small
// lattices an iteration is 7 launches of a few microseconds each and the solve is launch-bound otherwise.
// tsm_set_graphs(ctx, 0) turns it off.  Not used while per-launch profiling is on (events between the launches).
bool graphs_enabled(const tsm_ctx* ctx)
{
    return ctx->graphs_on != 0 && !ctx->prof_on && ctx->stream != nullptr && ctx->stream != cudaStreamLegacy && ctx->stream != cudaStreamPerThread;
}

bool cg_graph_cached(const tsm_ctx* ctx, int prec, int nrhs, int iters, const void* x, const void* r, const void* p, const void* w,
                     const void* t, double tol)
{
    for (const CgGraph& g : ctx->graphs)
        if (g.prec == prec && g.nrhs == nrhs && g.iters == iters && g.x == x && g.r == r && g.p == p && g.w == w && g.t == t && g.tol == tol)
            return true;
    return false;
}

int cg_iterations_graph(tsm_ctx* ctx, int prec, int nrhs, int iters, const Twists& tw, void* x, void* r, void* p, void* w, void* t, double tol)
{
    for (const CgGraph& g : ctx->graphs)
        if (g.prec == prec && g.nrhs == nrhs && g.iters == iters && g.x == x && g.r == r && g.p == p && g.w == w && g.t == t && g.tol == tol) {
            TSM_CUDA(ctx, cudaGraphLaunch(g.exec, ctx->stream));
            ctx->launches += g.launches;
            return TSM_OK;
        }
    const long long l0 = ctx->launches;
    TSM_CUDA(ctx, cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeRelaxed));
    int rc = TSM_OK;
    for (int k = 0; k < iters && rc == TSM_OK; k++) rc = cg_iteration(ctx, prec, nrhs, tw, x, r, p, w, t, tol);
    cudaGraph_t graph = nullptr;
    const cudaError_t e = cudaStreamEndCapture(ctx->stream, &graph);
    const long long in_graph = ctx->launches - l0;
    ctx->launches = l0;
    if (rc != TSM_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    TSM_CUDA(ctx, e);
    CgGraph g{prec, nrhs, iters, x, r, p, w, t, tol, in_graph, nullptr};
    const cudaError_t ei = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    TSM_CUDA(ctx, ei);
    if (ctx->graphs.size() >= 16) { cudaGraphExecDestroy(ctx->graphs.front().exec); ctx->graphs.erase(ctx->graphs.begin()); }
    ctx->graphs.push_back(g);
    TSM_CUDA(ctx, cudaGraphLaunch(g.exec, ctx->stream));
    ctx->launches += in_graph;
    return TSM_OK;
}

// The whole iteration loop as ONE graph launch: a WHILE node whose body is one captured CG iteration; the last
// block of k_cg_update_xp decides on the device whether another pass follows (sources left, cg->loop_left > 0).
// Residual mode then needs no host polling, and a solve on a small lattice is a handful of launches.
int cg_loop_graph(tsm_ctx* ctx, int prec, int nrhs, int n_iter, int eager, const Twists& tw, void* x, void* r, void* p, void* w, void* t,
                  double tol)
{
    int rc;
    if ((rc = launch_cg_loop_begin(ctx, n_iter))) return rc;
    ctx->loop_eager = eager;
    ctx->loop_nrhs = nrhs;
    for (const CgGraph& g : ctx->graphs)
        if (g.prec == prec && g.nrhs == nrhs && g.iters == 0 && g.x == x && g.r == r && g.p == p && g.w == w && g.t == t && g.tol == tol) {
            TSM_CUDA(ctx, cudaGraphLaunch(g.exec, ctx->stream));
            // one pass of the loop is counted here; the other passes (their number is known to the device only) are
            // added by fetch_scalars from the iteration counts
            ctx->launches += g.launches;
            ctx->loop_per_pass = g.launches;
            return TSM_OK;
        }
    cudaGraph_t graph = nullptr;
    TSM_CUDA(ctx, cudaGraphCreate(&graph, 0));
    cudaGraphConditionalHandle handle;
    cudaError_t e = cudaGraphConditionalHandleCreate(&handle, graph, 1, cudaGraphCondAssignDefault);
    cudaGraphNodeParams np = {};
    np.type = cudaGraphNodeTypeConditional;
    np.conditional.handle = handle;
    np.conditional.type = cudaGraphCondTypeWhile;
    np.conditional.size = 1;
    cudaGraphNode_t node;
    if (e == cudaSuccess) e = cudaGraphAddNode(&node, graph, nullptr, 0, &np);
    if (e != cudaSuccess) { cudaGraphDestroy(graph); TSM_CUDA(ctx, e); }
    cudaGraph_t body = np.conditional.phGraph_out[0];
    const long long l0 = ctx->launches;
    e = cudaStreamBeginCaptureToGraph(ctx->stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed);
    if (e != cudaSuccess) { cudaGraphDestroy(graph); TSM_CUDA(ctx, e); }
    rc = cg_iteration(ctx, prec, nrhs, tw, x, r, p, w, t, tol, (unsigned long long)handle, 1);
    e = cudaStreamEndCapture(ctx->stream, nullptr);
    const long long in_graph = ctx->launches - l0;
    ctx->launches = l0;
    if (rc != TSM_OK) { cudaGraphDestroy(graph); return rc; }
    if (e != cudaSuccess) { cudaGraphDestroy(graph); TSM_CUDA(ctx, e); }
    CgGraph g{prec, nrhs, 0, x, r, p, w, t, tol, in_graph, nullptr};
    e = cudaGraphInstantiate(&g.exec, graph, 0);
    cudaGraphDestroy(graph);
    TSM_CUDA(ctx, e);
    if (ctx->graphs.size() >= 16) { cudaGraphExecDestroy(ctx->graphs.front().exec); ctx->graphs.erase(ctx->graphs.begin()); }
    ctx->graphs.push_back(g);
    TSM_CUDA(ctx, cudaGraphLaunch(g.exec, ctx->stream));
    ctx->launches += in_graph;
    ctx->loop_per_pass = in_graph;
    return TSM_OK;
}

int fetch_scalars(tsm_ctx* ctx)
{
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->cg_host, ctx->cg, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    if (ctx->loop_per_pass > 0) {   // settle the launch count of the device-side loop that has just finished
        int most = 0;
        for (int j = 0; j < ctx->loop_nrhs; j++) most = ctx->cg_host->iters[j] > most ? ctx->cg_host->iters[j] : most;
        const int passes = most - ctx->loop_eager;
        if (passes > 1) ctx->launches += (long long)(passes - 1) * ctx->loop_per_pass;
        ctx->loop_per_pass = 0;
    }
    return TSM_OK;
}

// `max_iter` CG iterations at most, in chunks of 4; residual mode polls the all-done flag after each chunk.
int cg_run(tsm_ctx* ctx, int prec, int nrhs, const Twists& tw, void* x, void* r, void* p, void* w, void* t, double tol, int max_iter,
           bool no_poll = false)
{
    // iterations run in chunks of `poll`; in residual mode the host reads the all-done flag after each chunk
    // (a finished batch makes every later kernel return at once), in fixed-iteration mode it never does.
    // Full chunks run as one cached CUDA graph; the very first chunk of an argument set is launched kernel by
    // kernel (that also sets up the kernels' attributes, which must not happen inside a capture).
    int rc;
    const int poll = 4;
    const bool use_graph = graphs_enabled(ctx);
    // mode 3: the whole loop in ONE cooperative launch of k_cg_persistent (dslash.cu), where the lattice allows it
    // mode 4 (default): that launch where it measures faster (the lattices of k_dslash_small), graphs of 4 iterations elsewhere
    if (!ctx->prof_on && ((ctx->graphs_on == 3 && cg_persistent_supported(ctx, prec, nrhs)) ||
                          (ctx->graphs_on == 4 && cg_persistent_preferred(ctx, prec, nrhs)))) {
        const int rcp = launch_cg_persistent(ctx, prec, nrhs, x, r, p, w, t, {tw.zero, tw.Rinv}, {tw.R, tw.mk2}, {tw.zero, tw.Rbinv},
                                             {tw.Rb, tw.mk2}, tol, max_iter);
        if (rcp == TSM_OK || ctx->graphs_on == 3) return rcp;
        cudaGetLastError();   // automatic mode: a refused cooperative launch (nothing has run) falls back to the graph path
    }
    if (use_graph && (ctx->graphs_on == 2 || (no_poll && tol > 0))) {   // an enqueue-only solve in residual mode must not poll
        // device-side loop: the first iteration of an argument set runs kernel by kernel (kernel attributes
        // cannot be set inside a capture), everything after it is one graph launch
        int k = 0;
        if (!cg_graph_cached(ctx, prec, nrhs, 0, x, r, p, w, t, tol) && max_iter > 0) {
            if ((rc = cg_iteration(ctx, prec, nrhs, tw, x, r, p, w, t, tol))) return rc;
            k = 1;
        }
        if (k < max_iter) return cg_loop_graph(ctx, prec, nrhs, max_iter - k, k, tw, x, r, p, w, t, tol);
        return TSM_OK;
    }
    const bool cached = use_graph && cg_graph_cached(ctx, prec, nrhs, poll, x, r, p, w, t, tol);
    for (int k = 0; k < max_iter;) {
        const int chunk = max_iter - k < poll ? max_iter - k : poll;
        if (use_graph && (k > 0 || cached) && chunk == poll) {
            if ((rc = cg_iterations_graph(ctx, prec, nrhs, chunk, tw, x, r, p, w, t, tol))) return rc;
        } else {
            for (int j = 0; j < chunk; j++)
                if ((rc = cg_iteration(ctx, prec, nrhs, tw, x, r, p, w, t, tol))) return rc;
        }
        k += chunk;
        if (tol > 0 && k < max_iter) {
            TSM_CUDA(ctx, cudaMemcpyAsync(&ctx->cg_host->all_done, &ctx->cg->all_done, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
            TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
            if (ctx->cg_host->all_done) break;
        }
    }
    return TSM_OK;
}


// N4 (north_star "mixed-precision CG"): the HP solve as fp64 defect correction around the fp32
// CG.  On entry vec[0] = b' (fp64) and x64 is the slot's even half.  Loop: r = b' - A x in fp64 (the four
// stencil launches of an iteration, the last one with the residual epilogue and alpha = 1) -> stop when
// |r|/|b'| <= tol (A8, now the TRUE residual of the preconditioned normal system) -> e = fp32 CG on A e = r to
// MIXED_INNER_TOL -> x += e in fp64.  Every source has its own outer state and is frozen once converged (A14).
constexpr double MIXED_INNER_TOL = 1e-5;

int solve_mixed(tsm_ctx* ctx, int nrhs, const Twists& tw, void* x64, double tol, int max_iter)
{
    const int Vh = ctx->g.Vh;
    const size_t fb64 = field_bytes(TSM_F64, Vh, nrhs), fb32 = field_bytes(TSM_F32, Vh, nrhs);
    char* v0 = (char*)ctx->vec[0];
    void *R64 = ctx->vec[1], *b64 = ctx->vec[2], *w64 = ctx->vec[3], *t64 = ctx->vec[4];
    void *r32 = v0, *p32 = v0 + fb32, *w32 = ctx->vec[3], *t32 = (char*)ctx->vec[3] + fb32, *e32 = ctx->vec[5];
    int rc;
    TSM_CUDA(ctx, cudaMemcpyAsync(b64, ctx->vec[0], fb64, cudaMemcpyDeviceToDevice, ctx->stream));
    if ((rc = launch_cg_init(ctx, TSM_F64, nrhs, ctx->vec[0], R64, x64))) return rc;   // x = 0, R64 = b' = r(x = 0), |b'|^2
    if ((rc = launch_mixed_ctl(ctx, 0, nrhs, tol))) return rc;
    int prev[TSM_MAX_NRHS];
    for (int round = 0;; round++) {
        if ((rc = fetch_scalars(ctx))) return rc;
        const CgScalars sc = *ctx->cg_host;
        if (sc.all_outer_done) break;
        int most = 0;
        bool moved = round == 0;
        for (int j = 0; j < nrhs; j++) {
            if (!sc.outer_done[j] && sc.iters_outer[j] > most) most = sc.iters_outer[j];
            if (round > 0 && sc.iters_outer[j] != prev[j]) moved = true;
            prev[j] = sc.iters_outer[j];
        }
        if (most >= max_iter) break;   // TSM_ENOCONV for the live sources
        if (!moved) break;             // zero or broken-down inner systems: stop rather than spin
        if ((rc = launch_convert(ctx, TSM_F64, TSM_F32, nrhs, R64, r32))) return rc;
        if ((rc = launch_cg_init(ctx, TSM_F32, nrhs, r32, p32, e32))) return rc;
        if ((rc = launch_mixed_ctl(ctx, 1, nrhs, tol))) return rc;
        if ((rc = cg_run(ctx, TSM_F32, nrhs, tw, e32, r32, p32, w32, t32, MIXED_INNER_TOL, max_iter - most))) return rc;
        if ((rc = launch_mixed_ctl(ctx, 2, nrhs, tol))) return rc;
        if ((rc = launch_mixed_axpy(ctx, nrhs, x64, e32))) return rc;
        TSM_CUDA(ctx, cudaMemcpyAsync(R64, b64, fb64, cudaMemcpyDeviceToDevice, ctx->stream));
        if ((rc = launch_dslash(ctx, TSM_F64, 1, false, nrhs, x64, nullptr, t64, {tw.zero, tw.Rinv}, 0))) return rc;
        if ((rc = launch_dslash(ctx, TSM_F64, 0, false, nrhs, t64, x64, w64, {tw.R, tw.mk2}, 0))) return rc;
        if ((rc = launch_dslash(ctx, TSM_F64, 1, true, nrhs, w64, nullptr, t64, {tw.zero, tw.Rbinv}, 0))) return rc;
        if ((rc = launch_dslash(ctx, TSM_F64, 0, true, nrhs, t64, w64, R64, {tw.Rb, tw.mk2}, 4))) return rc;   // R64 = b' - A x
        if ((rc = launch_cg_reduce(ctx, 1, nrhs, 1))) return rc;
        if ((rc = launch_mixed_ctl(ctx, 3, nrhs, tol))) return rc;
    }
    return launch_mixed_ctl(ctx, 4, nrhs, tol);
}

// fp64 |eta - M s| / |eta| of the full system for every source of a slot (reading A8/A17).
int true_residuals(tsm_ctx* ctx, int slot, double* out)
{
    const int nrhs = ctx->slot_nrhs[slot], sp = ctx->slot_prec[slot];
    const size_t fb = field_bytes(TSM_F64, ctx->g.Vh, nrhs);
    // the six solver vectors are one contiguous region: three full-lattice fp64 fields
    char* base = (char*)ctx->vec[0];
    const size_t stride = 2 * ((char*)ctx->vec[1] - (char*)ctx->vec[0]);
    char *s64 = base, *eta = base + stride, *ms = base + 2 * stride;
    int rc;
    // convert both parities; a full field [parity][rhs] is 2*nrhs single-source parity fields
    if ((rc = launch_convert(ctx, sp, TSM_F64, 2 * nrhs, ctx->slot[slot], s64))) return rc;
    if ((rc = launch_noise(ctx, TSM_F64, nrhs, ctx->slot_seed[slot], ctx->ids_dev + slot * TSM_MAX_NRHS, ctx->slot_kind[slot], eta))) return rc;
    const Twists tw = make_twists(ctx);
    const TwistCoef mk = {-ctx->kappa, 0, -ctx->kappa, 0};
    if ((rc = launch_dslash(ctx, TSM_F64, 0, false, nrhs, s64 + fb, s64, ms, {tw.R, mk}, 0))) return rc;
    if ((rc = launch_dslash(ctx, TSM_F64, 1, false, nrhs, s64, s64 + fb, ms + fb, {tw.R, mk}, 0))) return rc;
    if ((rc = launch_diff_norm2(ctx, nrhs, eta, ms))) return rc;
    if ((rc = fetch_scalars(ctx))) return rc;
    const double eta2 = 12.0 * (double)ctx->g.V;   // |eta_{alpha c}(x)| = 1 for Z4 and Z2
    for (int j = 0; j < nrhs; j++) out[j] = std::sqrt(ctx->cg_host->pq[j] / eta2);
    return TSM_OK;
}

int check_loops(tsm_ctx* ctx)
{
    if (!ctx->loops_ready) return tsm_fail(ctx, TSM_ESTATE, "loop accumulators not set up: call tsm_loops_reset (also after tsm_loops_set_momenta)");
    return TSM_OK;
}

int check_slot(tsm_ctx* ctx, int slot, int rhs)
{
    if (slot < 0 || slot > 1) return tsm_fail(ctx, TSM_EINVAL, "slot must be 0 or 1");
    if (ctx->slot_prec[slot] < 0) return tsm_fail(ctx, TSM_ESTATE, "slot holds no solution");
    if (rhs < 0 || rhs >= ctx->slot_nrhs[slot]) return tsm_fail(ctx, TSM_EINVAL, "rhs out of range for this slot");
    return TSM_OK;
}

// Everything a solve puts on the stream: noise, source preparation, CG, reconstruction, and a pinned snapshot of the
// CG scalars for solve_collect.  no_poll: never synchronise with the host (residual mode then runs the device-side
// iteration loop; the mixed-precision solver still reads its outer-loop state on the host).
int solve_enqueue(tsm_ctx* ctx, uint64_t seed, const uint32_t* source_ids, int nrhs, int kind, int prec, double tol, int max_iter, int slot,
                  bool no_poll)
{
    int rc = ctx_enter(ctx, true, true, true);
    if (rc) return rc;
    if (!source_ids || nrhs < 1 || nrhs > ctx->max_nrhs || (kind != TSM_Z4 && kind != TSM_Z2) || prec < 0 || prec > TSM_MIXED ||
        !(tol >= 0) || max_iter < 0 || slot < 0 || slot > 1 || (prec == TSM_MIXED && !(tol > 0)))
        return tsm_fail(ctx, TSM_EINVAL, "bad solve arguments");
    if (ctx->ws_prec != TSM_F64 && (prec == TSM_F64 || prec == TSM_MIXED))
        return tsm_fail(ctx, TSM_ESTATE, "fp64 solve on a low-precision-only workspace (tsm_set_workspace prec)");
    // bf16 storage (config 4): source preparation, x, r, q, reconstruction and the stored solution are
    // fp32; only the search direction p and the stencil temporaries t, w are bf16 (fp32 arithmetic).
    const int sp = prec == TSM_BF16 ? TSM_F32 : (prec == TSM_MIXED ? TSM_F64 : prec);   // precision of the stored solution
    const int Vh = ctx->g.Vh;
    const Twists tw = make_twists(ctx);
    ctx->slot_prec[slot] = sp;
    ctx->slot_nrhs[slot] = nrhs;
    ctx->slot_kind[slot] = kind;
    ctx->slot_seed[slot] = seed;
    memcpy(ctx->slot_ids[slot], source_ids, nrhs * sizeof(uint32_t));
    uint32_t* ids_dev = ctx->ids_dev + slot * TSM_MAX_NRHS;
    TSM_CUDA(ctx, cudaMemcpyAsync(ids_dev, ctx->slot_ids[slot], nrhs * sizeof(uint32_t), cudaMemcpyHostToDevice, ctx->stream));
    TSM_CUDA(ctx, cudaEventRecord(ctx->slot_ev0[slot], ctx->stream));
    ctx->loop_per_pass = 0;

    char* s_e = (char*)ctx->slot[slot];
    char* s_o = s_e + field_bytes(sp, Vh, nrhs);
    void *r = ctx->vec[0], *p = ctx->vec[1], *w = ctx->vec[3], *t = ctx->vec[4], *aux = ctx->vec[5];
    void* x = s_e;
    {   // H3: eta straight into the slot (eta_e where s_e will be, eta_o where s_o will be)
        Phase ph("tsm: noise");
        if ((rc = launch_noise(ctx, sp, nrhs, seed, ids_dev, kind, s_e))) return rc;
    }
    // Automatic launch mode on the smallest lattices: everything after the noise in ONE cooperative launch (dslash_small.cu:
    // k_cg_persistent_small in its whole-solve form; the same arithmetic in the same order as the steps below)
    bool one_launch = false;
    if (prec != TSM_MIXED && prec != TSM_BF16 && ctx->graphs_on == 4 && !ctx->prof_on && cg_persistent_preferred(ctx, prec, nrhs)) {
        Phase ph("tsm: prepare + CG + reconstruct (one launch)");
        PcgArgs wa{};
        wa.s_o = s_o; wa.aux = aux; wa.tw_rinv = tw.Rinv;
        wa.cp1 = {tw.one, tw.k}; wa.cp2 = {tw.zero, tw.Rbinv}; wa.cp3 = {tw.Rb, tw.mk2}; wa.crec = {tw.Rinv, tw.kRinv};
        const int rcw = launch_cg_persistent(ctx, prec, nrhs, x, r, p, w, t, {tw.zero, tw.Rinv}, {tw.R, tw.mk2}, {tw.zero, tw.Rbinv},
                                             {tw.Rb, tw.mk2}, tol, max_iter, &wa);
        if (rcw == TSM_OK) one_launch = true;
        else cudaGetLastError();   // refused (nothing has run): the step-by-step path below
    }
    if (!one_launch) {   // H4: bhat = eta_e + kappa D_eo R^-1 eta_o (into w);  b' = Mhat^dag bhat (into r)
        Phase ph("tsm: prepare");
        if ((rc = launch_twist(ctx, sp, nrhs, s_o, aux, tw.Rinv))) return rc;
        if ((rc = launch_dslash(ctx, sp, 0, false, nrhs, aux, s_e, w, {tw.one, tw.k}, 0))) return rc;
        if ((rc = launch_dslash(ctx, sp, 1, true, nrhs, w, nullptr, t, {tw.zero, tw.Rbinv}, 0))) return rc;
        if ((rc = launch_dslash(ctx, sp, 0, true, nrhs, t, w, r, {tw.Rb, tw.mk2}, 0))) return rc;
    }
    if (!one_launch) {   // O5: x0 = 0 (x lives in the slot's even half), r0 = p0 = b'
        Phase ph(prec == TSM_MIXED ? "tsm: CG (mixed precision)" : "tsm: CG");
        if (prec == TSM_MIXED) {
            if ((rc = solve_mixed(ctx, nrhs, tw, s_e, tol, max_iter))) return rc;
        } else {
            if ((rc = launch_cg_init(ctx, prec, nrhs, r, p, x))) return rc;
            if ((rc = cg_run(ctx, prec, nrhs, tw, x, r, p, w, t, tol, max_iter, no_poll))) return rc;
        }
    }
    if (!one_launch) {   // H7: s_e = x, s_o = R^-1 (eta_o + kappa D_oe x)
        Phase ph("tsm: reconstruct");
        if ((rc = launch_dslash(ctx, sp, 1, false, nrhs, x, s_o, aux, {tw.Rinv, tw.kRinv}, 0))) return rc;
        TSM_CUDA(ctx, cudaMemcpyAsync(s_o, aux, field_bytes(sp, Vh, nrhs), cudaMemcpyDeviceToDevice, ctx->stream));
    }
    TSM_CUDA(ctx, cudaEventRecord(ctx->slot_ev1[slot], ctx->stream));
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->cg_snap[slot], ctx->cg, sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream));
    ctx->slot_tol[slot] = tol;
    ctx->slot_pending[slot] = true;
    ctx->slot_loop_per_pass[slot] = ctx->loop_per_pass;   // a device-side loop of this solve whose passes are not yet counted
    ctx->slot_loop_eager[slot] = ctx->loop_eager;
    ctx->loop_per_pass = 0;
    return TSM_OK;
}

// Waits for the solve last enqueued into `slot` and reports on it (iteration counts, status, residuals, time).
int solve_collect(tsm_ctx* ctx, int slot, int want_true_resid, tsm_solve_info* info)
{
    int rc;
    if (slot < 0 || slot > 1 || !ctx->slot_pending[slot]) return tsm_fail(ctx, TSM_ESTATE, "no solve is pending on this slot");
    if (want_true_resid && ctx->ws_prec != TSM_F64)
        return tsm_fail(ctx, TSM_ESTATE, "fp64 true residual on a low-precision-only workspace (tsm_set_workspace prec)");
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->slot_pending[slot] = false;
    const CgScalars sc = *ctx->cg_snap[slot];
    const int nrhs = ctx->slot_nrhs[slot];
    const double tol = ctx->slot_tol[slot];
    if (ctx->slot_loop_per_pass[slot] > 0) {   // settle the launch count of the solve's device-side loop
        int most = 0;
        for (int j = 0; j < nrhs; j++) most = sc.iters[j] > most ? sc.iters[j] : most;
        const int passes = most - ctx->slot_loop_eager[slot];
        if (passes > 1) ctx->launches += (long long)(passes - 1) * ctx->slot_loop_per_pass[slot];
        ctx->slot_loop_per_pass[slot] = 0;
    }
    float ms = 0;
    TSM_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->slot_ev0[slot], ctx->slot_ev1[slot]));
    double tr[TSM_MAX_NRHS];
    for (int j = 0; j < nrhs; j++) tr[j] = -1.0;
    if (want_true_resid && (rc = true_residuals(ctx, slot, tr))) return rc;
    int first = TSM_OK;
    for (int j = 0; j < nrhs; j++) {
        int st = sc.status[j];
        if (st == TSM_OK && tol > 0 && !sc.done[j]) st = TSM_ENOCONV;
        if (first == TSM_OK && st != TSM_OK) first = st;
        if (info) {
            info[j].iters = sc.iters[j];
            info[j].status = st;
            info[j].rel_resid_rec = sc.bb[j] > 0 ? std::sqrt(sc.rr[j] / sc.bb[j]) : 0.0;
            info[j].rel_resid_true = tr[j];
            info[j].secs = ms * 1e-3;
        }
    }
    if (first != TSM_OK) ctx->err = first == TSM_ENOCONV ? "tolerance not reached in max_iter" : "CG breakdown";
    return first;
}

}  // namespace

extern "C" {

int tsm_solve(tsm_ctx* ctx, uint64_t seed, const uint32_t* source_ids, int nrhs, int kind, int prec, double tol,
              int max_iter, int slot, int want_true_resid, tsm_solve_info* info)
{
    if (ctx && want_true_resid && ctx->ws_prec != TSM_F64)
        return tsm_fail(ctx, TSM_ESTATE, "fp64 true residual on a low-precision-only workspace (tsm_set_workspace prec)");
    const int rc = solve_enqueue(ctx, seed, source_ids, nrhs, kind, prec, tol, max_iter, slot, false);
    if (rc) return rc;
    return solve_collect(ctx, slot, want_true_resid, info);
}

int tsm_solve_async(tsm_ctx* ctx, uint64_t seed, const uint32_t* source_ids, int nrhs, int kind, int prec, double tol,
                    int max_iter, int slot)
{
    return solve_enqueue(ctx, seed, source_ids, nrhs, kind, prec, tol, max_iter, slot, true);
}

int tsm_solve_wait(tsm_ctx* ctx, int slot, int want_true_resid, tsm_solve_info* info)
{
    const int rc = ctx_enter(ctx, true, true, true);
    if (rc) return rc;
    return solve_collect(ctx, slot, want_true_resid, info);
}

int tsm_get_solution(tsm_ctx* ctx, int slot, int rhs, double* host_out)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if ((rc = check_slot(ctx, slot, rhs))) return rc;
    if (!host_out) return tsm_fail(ctx, TSM_EINVAL, "null output");
    const int sp = ctx->slot_prec[slot], nrhs = ctx->slot_nrhs[slot], Vh = ctx->g.Vh;
    // unpack the two parities of source `rhs` straight from the slot (parity stride = the slot's [rhs] extent)
    const char* src = (const char*)ctx->slot[slot] + field_bytes(sp, Vh, 1) * rhs;
    if ((rc = launch_unpack_spinor(ctx, sp, 1, src, (double*)ctx->staging, field_bytes(sp, Vh, nrhs)))) return rc;
    TSM_CUDA(ctx, cudaMemcpyAsync(host_out, ctx->staging, (size_t)ctx->g.V * 24 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return TSM_OK;
}

int tsm_set_solution(tsm_ctx* ctx, int slot, int rhs, const double* host_in)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if ((rc = check_slot(ctx, slot, rhs))) return rc;
    if (!host_in) return tsm_fail(ctx, TSM_EINVAL, "null input");
    const int sp = ctx->slot_prec[slot], nrhs = ctx->slot_nrhs[slot], Vh = ctx->g.Vh;
    char* dst = (char*)ctx->slot[slot] + field_bytes(sp, Vh, 1) * rhs;
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->staging, host_in, (size_t)ctx->g.V * 24 * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    if ((rc = launch_pack_spinor(ctx, sp, 1, (const double*)ctx->staging, dst, field_bytes(sp, Vh, nrhs)))) return rc;
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return TSM_OK;
}

int tsm_loops_reset(tsm_ctx* ctx, int ops)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if (ops < 0 || ops > (TSM_OPS_DERIVATIVE | TSM_OPS_ONE_END | TSM_OPS_GEN_ONE_END | TSM_OPS_MOMENTA))
        return tsm_fail(ctx, TSM_EINVAL, "bad loop operator set");
    ctx->with_deriv = (ops & TSM_OPS_DERIVATIVE) ? 1 : 0;
    ctx->with_one_end = (ops & TSM_OPS_ONE_END) ? 1 : 0;
    ctx->with_gen_one_end = (ops & TSM_OPS_GEN_ONE_END) ? 1 : 0;
    ctx->n_ops = TSM_N_LOCAL_OPS + (ctx->with_deriv ? TSM_N_DERIV_OPS : 0) + (ctx->with_one_end ? TSM_N_ONE_END_OPS : 0) +
                 (ctx->with_gen_one_end ? TSM_N_GEN_ONE_END_OPS : 0);
    ctx->with_momenta = (ops & TSM_OPS_MOMENTA) ? 1 : 0;
    if (ctx->with_momenta) ctx->n_ops += 16 * ctx->n_mom;
    ctx->n_hp = ctx->n_lp = 0;
    const size_t lb = (size_t)ctx->n_ops * ctx->g.L[3] * 2 * sizeof(double);
    TSM_CUDA(ctx, cudaMemsetAsync(ctx->acc_corr, 0, lb, ctx->stream));
    TSM_CUDA(ctx, cudaMemsetAsync(ctx->acc_lp, 0, lb, ctx->stream));
    ctx->loops_ready = true;
    return TSM_OK;
}

int tsm_set_graphs(tsm_ctx* ctx, int mode)
{
    if (!ctx) return TSM_EINVAL;
    if (mode < 0 || mode > 4)
        return tsm_fail(ctx, TSM_EINVAL, "graphs: 0 off, 1 chunks of 4 iterations, 2 device-side loop, 3 persistent cooperative kernel, 4 automatic");
    ctx->graphs_on = mode;
    return TSM_OK;
}

int tsm_set_hp_precision(tsm_ctx* ctx, int prec)
{
    if (!ctx) return TSM_EINVAL;
    if (prec != TSM_F64 && prec != TSM_MIXED) return tsm_fail(ctx, TSM_EINVAL, "HP precision must be TSM_F64 or TSM_MIXED");
    ctx->hp_prec = prec;
    return TSM_OK;
}

int tsm_loops_set_momenta(tsm_ctx* ctx, int nmom, const int* n)
{
    if (!ctx) return TSM_EINVAL;
    if (nmom < 0 || nmom > TSM_MAX_MOMENTA || (nmom > 0 && !n)) return tsm_fail(ctx, TSM_EINVAL, "bad momentum list");
    ctx->n_mom = nmom;
    ctx->loops_ready = false;   // n_ops and the accumulators' shape are fixed by the next tsm_loops_reset
    for (int m = 0; m < nmom; m++)
        for (int k = 0; k < 3; k++) ctx->mom[m][k] = n[3 * m + k];
    return TSM_OK;
}

int tsm_loops_add_correction(tsm_ctx* ctx, int slot_hp, int slot_lp)
{
    int rc = ctx_enter(ctx, true, true, false);
    if (rc) return rc;
    if ((rc = check_loops(ctx))) return rc;
    if ((rc = check_slot(ctx, slot_hp, 0)) || (rc = check_slot(ctx, slot_lp, 0))) return rc;
    if (slot_hp == slot_lp) return tsm_fail(ctx, TSM_EINVAL, "HP and LP slots must differ");
    const int nrhs = ctx->slot_nrhs[slot_hp];
    if (nrhs != ctx->slot_nrhs[slot_lp] || ctx->slot_seed[slot_hp] != ctx->slot_seed[slot_lp] ||
        ctx->slot_kind[slot_hp] != ctx->slot_kind[slot_lp] ||
        memcmp(ctx->slot_ids[slot_hp], ctx->slot_ids[slot_lp], nrhs * sizeof(uint32_t)) != 0)
        return tsm_fail(ctx, TSM_ESTATE, "HP and LP slots hold different sources (Eq. 2.4 needs the same eta_j)");
    Phase ph("tsm: contract (HP - LP)");
    if ((rc = launch_contract(ctx, slot_hp))) return rc;
    if ((rc = launch_contract(ctx, slot_lp))) return rc;
    if ((rc = launch_accumulate(ctx, ctx->acc_corr, ctx->loops_src[slot_hp], ctx->loops_src[slot_lp], nrhs))) return rc;
    ctx->n_hp += nrhs;
    return TSM_OK;
}

int tsm_loops_add_lp(tsm_ctx* ctx, int slot_lp)
{
    int rc = ctx_enter(ctx, true, true, false);
    if (rc) return rc;
    if ((rc = check_loops(ctx))) return rc;
    if ((rc = check_slot(ctx, slot_lp, 0))) return rc;
    const int nrhs = ctx->slot_nrhs[slot_lp];
    Phase ph("tsm: contract (LP)");
    if ((rc = launch_contract(ctx, slot_lp))) return rc;
    if ((rc = launch_accumulate(ctx, ctx->acc_lp, ctx->loops_src[slot_lp], nullptr, nrhs))) return rc;
    ctx->n_lp += nrhs;
    return TSM_OK;
}

int tsm_loops_source(tsm_ctx* ctx, int slot, int rhs, double* host_out)
{
    int rc = ctx_enter(ctx, true, true, false);
    if (rc) return rc;
    if ((rc = check_loops(ctx))) return rc;
    if ((rc = check_slot(ctx, slot, rhs))) return rc;
    if (!host_out) return tsm_fail(ctx, TSM_EINVAL, "null output");
    if ((rc = launch_contract(ctx, slot))) return rc;
    const size_t lb = (size_t)ctx->n_ops * ctx->g.L[3] * 2 * sizeof(double);
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->host_small, (char*)ctx->loops_src[slot] + lb * rhs, lb, cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    memcpy(host_out, ctx->host_small, lb);
    return TSM_OK;
}

int tsm_loops_finalize(tsm_ctx* ctx, double* host_out)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if (!host_out) return tsm_fail(ctx, TSM_EINVAL, "null output");
    if ((rc = check_loops(ctx))) return rc;
    if ((rc = launch_finalize(ctx))) return rc;
    const size_t lb = (size_t)ctx->n_ops * ctx->g.L[3] * 2 * sizeof(double);
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->host_small, ctx->loops_out, lb, cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    memcpy(host_out, ctx->host_small, lb);
    return TSM_OK;
}

int tsm_loops_get_state(tsm_ctx* ctx, double* host_corr, double* host_lp, int* n_hp, int* n_lp)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if (!host_corr || !host_lp || !n_hp || !n_lp) return tsm_fail(ctx, TSM_EINVAL, "null output");
    if ((rc = check_loops(ctx))) return rc;
    const size_t lb = (size_t)ctx->n_ops * ctx->g.L[3] * 2 * sizeof(double);
    TSM_CUDA(ctx, cudaMemcpyAsync(host_corr, ctx->acc_corr, lb, cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaMemcpyAsync(host_lp, ctx->acc_lp, lb, cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    *n_hp = ctx->n_hp;
    *n_lp = ctx->n_lp;
    return TSM_OK;
}

int tsm_loops_set_state(tsm_ctx* ctx, const double* host_corr, const double* host_lp, int n_hp, int n_lp)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if (!host_corr || !host_lp || n_hp < 0 || n_lp < 0) return tsm_fail(ctx, TSM_EINVAL, "bad state");
    if ((rc = check_loops(ctx))) return rc;
    const size_t lb = (size_t)ctx->n_ops * ctx->g.L[3] * 2 * sizeof(double);
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->acc_corr, host_corr, lb, cudaMemcpyHostToDevice, ctx->stream));
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->acc_lp, host_lp, lb, cudaMemcpyHostToDevice, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    ctx->n_hp = n_hp;
    ctx->n_lp = n_lp;
    return TSM_OK;
}

int tsm_run_loop_set(tsm_ctx* ctx, uint64_t seed, int kind, int n_hp, int n_lp, int lp_prec, double lp_tol, int lp_iters,
                     double hp_tol, int hp_max_iter, int nrhs, int ops, double* host_out, double* secs_out)
{
    int rc = ctx_enter(ctx, true, true, true);
    if (rc) return rc;
    if (n_hp < 0 || n_lp < 0 || nrhs < 1 || nrhs > ctx->max_nrhs || !host_out) return tsm_fail(ctx, TSM_EINVAL, "bad loop-set arguments");
    cudaEvent_t e0, e1;
    TSM_CUDA(ctx, cudaEventCreate(&e0));
    TSM_CUDA(ctx, cudaEventCreate(&e1));
    TSM_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
    int worst = TSM_OK;
    if ((rc = tsm_loops_reset(ctx, ops))) goto fail;
    for (int j0 = 0; j0 < n_hp + n_lp;) {
        const bool hp = j0 < n_hp;
        // the HP batches are waited for one by one (their status is known); the sticky flag only has to cover the
        // LP-only batches that follow (an inner fp32 CG of the mixed-precision HP solver may set it harmlessly)
        if (j0 == n_hp && cudaMemsetAsync(&ctx->cg->sticky_breakdown, 0, sizeof(int), ctx->stream) != cudaSuccess) { rc = TSM_ECUDA; goto fail; }
        const int end = hp ? n_hp : n_hp + n_lp;
        const int nb = (end - j0 < nrhs) ? end - j0 : nrhs;
        uint32_t ids[TSM_MAX_NRHS];
        for (int k = 0; k < nb; k++) ids[k] = (uint32_t)(j0 + k);
        if (hp) {
            rc = tsm_solve(ctx, seed, ids, nb, kind, ctx->hp_prec, hp_tol, hp_max_iter, 0, 0, nullptr);
            if (rc == TSM_ECUDA || rc == TSM_EINVAL || rc == TSM_ESTATE) goto fail;
            if (rc && !worst) worst = rc;
        }
        if (hp) {
            rc = tsm_solve(ctx, seed, ids, nb, kind, lp_prec, lp_tol, lp_iters, 1, 0, nullptr);
            // an LP solve that hits its iteration cap is still a valid truncated estimate
            if (rc == TSM_ECUDA || rc == TSM_EINVAL || rc == TSM_ESTATE) goto fail;
            if (rc == TSM_EBREAKDOWN && !worst) worst = rc;
        } else {
            // LP-only batches are only enqueued: the host runs ahead of the device (on small lattices a solve is a few
            // dozen launches of a few microseconds); a breakdown in any of them is read from a sticky flag at the end
            rc = tsm_solve_async(ctx, seed, ids, nb, kind, lp_prec, lp_tol, lp_iters, 1);
            if (rc) goto fail;
        }
        rc = hp ? tsm_loops_add_correction(ctx, 0, 1) : tsm_loops_add_lp(ctx, 1);
        if (rc) goto fail;
        j0 += nb;
    }
    if ((rc = launch_finalize(ctx))) goto fail;
    TSM_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
    if ((rc = fetch_scalars(ctx))) goto fail;
    ctx->slot_pending[1] = false;
    if (n_lp > 0 && ctx->cg_host->sticky_breakdown && !worst) worst = TSM_EBREAKDOWN;
    if ((rc = tsm_loops_finalize(ctx, host_out))) goto fail;
    if (secs_out) {
        float ms = 0;
        TSM_CUDA(ctx, cudaEventElapsedTime(&ms, e0, e1));
        *secs_out = ms * 1e-3;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return worst;
fail:
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return rc;
}

}  // extern "C"
