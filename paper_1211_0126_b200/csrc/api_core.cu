// api_core.cu -- C ABI (include/tsm.h): context, workspace carving, gauge ingest, layout
// conversion, noise hook and the single-application stencil entry.
#include <cmath>
#include <cstring>
#include <new>

#include "tsm_internal.cuh"

namespace {

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Carve {
    size_t off = 0;
    size_t take(size_t bytes) { const size_t o = off; off = align256(off + bytes); return o; }
};

// One place that defines the workspace layout; used both to size it and to carve it.
// prec: TSM_F64 = everything (fp64 link packs, fp64-sized vectors and slots); TSM_F32 = a low-precision-only
// workspace (fp32 / bf16 solves: no fp64 link packs, vectors and slots sized for fp32 fields).
size_t carve_workspace(tsm_ctx* ctx, int max_nrhs, int prec, char* base)
{
    const Geom& g = ctx->g;
    Carve c;
    auto at = [&](size_t o) -> void* { return base ? base + o : nullptr; };
    const bool wide = prec == TSM_F64;
    if (base) ctx->gauge64[0] = ctx->gauge64[1] = nullptr;
    if (wide)
        for (int p = 0; p < 2; p++) { size_t o = c.take(gauge_pack_bytes(1, 18, g.Vh)); if (base) ctx->gauge64[p] = at(o); }
    for (int p = 0; p < 2; p++) { size_t o = c.take(gauge_pack_bytes(0, 18, g.Vh)); if (base) ctx->gauge32[p] = at(o); }
    size_t stg = (size_t)4 * g.V * 18 * sizeof(double);
    const size_t stg2 = (size_t)max_nrhs * g.V * 24 * sizeof(double);
    if (stg2 > stg) stg = stg2;
    { size_t o = c.take(stg); if (base) { ctx->staging = at(o); ctx->staging_bytes = stg; } }
    const size_t fb = align256(field_bytes(wide ? TSM_F64 : TSM_F32, g.Vh, max_nrhs));
    { size_t o = c.take(6 * fb); if (base) for (int k = 0; k < 6; k++) ctx->vec[k] = at(o + k * fb); }
    for (int s = 0; s < 2; s++) { size_t o = c.take(2 * fb); if (base) ctx->slot[s] = at(o); }
    size_t pc = (size_t)ctx->nsm * 16 * max_nrhs;
    const size_t pc2 = (size_t)max_nrhs * (7 + TSM_MAX_MOMENTA) * g.L[3] * 2 * 8 * 32;
    if (pc2 > pc) pc = pc2;
    { size_t o = c.take(pc * sizeof(double)); if (base) { ctx->partials = (double*)at(o); ctx->partials_count = pc; } }
    const size_t npc = (size_t)max_nrhs * ((g.Vh + 127) / 128) * 8;   // per (source, tile): one partial, or one per warp of the box stencil
    { size_t o = c.take(npc * sizeof(double)); if (base) { ctx->norm_partials = (double*)at(o); ctx->norm_partials_count = npc; } }
    const size_t lb = (size_t)TSM_MAX_OPS * g.L[3] * 2 * sizeof(double);
    for (int s = 0; s < 2; s++) { size_t o = c.take(lb * max_nrhs); if (base) ctx->loops_src[s] = (double*)at(o); }
    { size_t o = c.take(lb); if (base) ctx->acc_corr = (double*)at(o); }
    { size_t o = c.take(lb); if (base) ctx->acc_lp = (double*)at(o); }
    { size_t o = c.take(lb); if (base) ctx->loops_out = (double*)at(o); }
    return c.off;
}

}  // namespace

int ctx_enter(tsm_ctx* ctx, bool need_ws, bool need_gauge, bool need_params)
{
    if (!ctx) return TSM_EINVAL;
    TSM_CUDA(ctx, cudaSetDevice(ctx->device));
    if (need_ws && !ctx->have_ws) return tsm_fail(ctx, TSM_ESTATE, "no workspace set (tsm_set_workspace)");
    if (need_gauge && !ctx->have_gauge) return tsm_fail(ctx, TSM_ESTATE, "no gauge field set (tsm_set_gauge)");
    if (need_params && !ctx->have_params) return tsm_fail(ctx, TSM_ESTATE, "kappa/mu not set (tsm_set_params)");
    return TSM_OK;
}

void ctx_drop_graphs(tsm_ctx* ctx)
{
    for (CgGraph& g : ctx->graphs) cudaGraphExecDestroy(g.exec);
    ctx->graphs.clear();
}

extern "C" {

int tsm_create(tsm_ctx** out, const int dims[4], int t_boundary, int device)
{
    if (!out || !dims) return TSM_EINVAL;
    *out = nullptr;
    for (int k = 0; k < 4; k++)
        if (dims[k] < 4 || (dims[k] & 1)) return TSM_EINVAL;
    if (t_boundary != 1 && t_boundary != -1) return TSM_EINVAL;
    const long long V = (long long)dims[0] * dims[1] * dims[2] * dims[3];
    if (V / 2 > 0x3fffffffLL) return TSM_EINVAL;   // cb indices are 32-bit
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return TSM_ECUDA;
    tsm_ctx* ctx = new (std::nothrow) tsm_ctx();
    if (!ctx) return TSM_ECUDA;
    for (int k = 0; k < 4; k++) ctx->g.L[k] = dims[k];
    ctx->g.Lxh = dims[0] / 2;
    ctx->g.Vsh = dims[0] * dims[1] * dims[2] / 2;
    ctx->g.V = V;
    ctx->g.Vh = (int)(V / 2);
    ctx->g.theta = t_boundary;
    {   // traversal slabs: the largest divisor of Lz that is <= 8 z-planes
        Geom& g = ctx->g;
        g.S = g.Lxh * dims[1];
        g.bz = 1;
        for (int b = 1; b <= 8 && b <= dims[2]; b++)
            if (dims[2] % b == 0) g.bz = b;
        g.dLxh = make_fastdiv(g.Lxh); g.dLy = make_fastdiv(dims[1]); g.dLz = make_fastdiv(dims[2]);
        g.dS = make_fastdiv(g.S); g.dSB = make_fastdiv(g.bz * g.S); g.dLt = make_fastdiv(dims[3]);
    }
    ctx->device = device;
    ctx->stream = 0;
    ctx->own_stream = nullptr;
    ctx->have_params = ctx->have_gauge = ctx->have_ws = false;
    ctx->recon = 18;
    ctx->max_nrhs = 0;
    ctx->norm_reduced = false;
    ctx->ws_prec = TSM_F64;
    ctx->n_ops = TSM_N_LOCAL_OPS;
    ctx->with_deriv = 0;
    ctx->with_one_end = 0;
    ctx->with_gen_one_end = 0;
    ctx->with_momenta = 0;
    ctx->hp_prec = TSM_MIXED;
    ctx->n_mom = 0;
    ctx->n_hp = ctx->n_lp = 0;
    ctx->launches = 0;
    ctx->prof_on = false;
    ctx->loops_ready = false;
    ctx->stencil_choice = 0;
    ctx->graphs_on = 4;
    ctx->loop_per_pass = 0;
    ctx->cg = nullptr; ctx->cg_host = nullptr; ctx->host_small = nullptr; ctx->ids_dev = nullptr;
    for (int s = 0; s < 2; s++) { ctx->slot_prec[s] = -1; ctx->slot_nrhs[s] = 0; }
    build_gamma_table(ctx->gam);
    bool ok = cudaSetDevice(device) == cudaSuccess;
    cudaDeviceProp prop;
    ok = ok && cudaGetDeviceProperties(&prop, device) == cudaSuccess;
    if (ok) ctx->nsm = prop.multiProcessorCount;
    ok = ok && cudaMalloc(&ctx->cg, sizeof(CgScalars)) == cudaSuccess;
    ok = ok && cudaMemset(ctx->cg, 0, sizeof(CgScalars)) == cudaSuccess;
    ok = ok && cudaMallocHost(&ctx->cg_host, sizeof(CgScalars)) == cudaSuccess;
    for (int s = 0; s < 2; s++) {
        ctx->cg_snap[s] = nullptr; ctx->slot_ev0[s] = ctx->slot_ev1[s] = nullptr; ctx->slot_pending[s] = false; ctx->slot_loop_per_pass[s] = 0;
        ok = ok && cudaMallocHost(&ctx->cg_snap[s], sizeof(CgScalars)) == cudaSuccess;
        ok = ok && cudaEventCreate(&ctx->slot_ev0[s]) == cudaSuccess && cudaEventCreate(&ctx->slot_ev1[s]) == cudaSuccess;
    }
    const size_t hs = (size_t)TSM_MAX_OPS * dims[3] * 2 * sizeof(double) * 2 + 256;
    ok = ok && cudaMallocHost(&ctx->host_small, hs) == cudaSuccess;
    ok = ok && cudaMalloc(&ctx->ids_dev, 2 * TSM_MAX_NRHS * sizeof(uint32_t)) == cudaSuccess;
    ok = ok && cudaEventCreate(&ctx->ev0) == cudaSuccess && cudaEventCreate(&ctx->ev1) == cudaSuccess;
    ok = ok && cudaStreamCreate(&ctx->own_stream) == cudaSuccess;   // blocking: ordered with the legacy default stream
    ctx->stream = ctx->own_stream;
    if (!ok) { tsm_destroy(ctx); return TSM_ECUDA; }
    *out = ctx;
    return TSM_OK;
}

int tsm_destroy(tsm_ctx* ctx)
{
    if (!ctx) return TSM_EINVAL;
    cudaSetDevice(ctx->device);
    ctx_drop_graphs(ctx);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    if (ctx->cg) cudaFree(ctx->cg);
    if (ctx->cg_host) cudaFreeHost(ctx->cg_host);
    for (int s = 0; s < 2; s++) {
        if (ctx->cg_snap[s]) cudaFreeHost(ctx->cg_snap[s]);
        if (ctx->slot_ev0[s]) cudaEventDestroy(ctx->slot_ev0[s]);
        if (ctx->slot_ev1[s]) cudaEventDestroy(ctx->slot_ev1[s]);
    }
    if (ctx->host_small) cudaFreeHost(ctx->host_small);
    if (ctx->ids_dev) cudaFree(ctx->ids_dev);
    for (ProfRec& r : ctx->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (cudaEvent_t e : ctx->prof_pool) cudaEventDestroy(e);
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    delete ctx;
    return TSM_OK;
}

const char* tsm_last_error(const tsm_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

long long tsm_launch_count(const tsm_ctx* ctx) { return ctx ? ctx->launches : 0; }

int tsm_profile(tsm_ctx* ctx, int enable)
{
    if (!ctx) return TSM_EINVAL;
    ctx->prof_on = enable != 0;
    return TSM_OK;
}

int tsm_profile_read(tsm_ctx* ctx, int prec, int kind, int nrhs, double* total_ms, long long* count)
{
    if (!ctx || !total_ms || !count) return TSM_EINVAL;
    TSM_CUDA(ctx, cudaSetDevice(ctx->device));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    double tot = 0;
    long long n = 0;
    std::vector<ProfRec> keep;
    for (ProfRec& r : ctx->prof) {
        if (r.prec == prec && r.kind == kind && (nrhs <= 0 || r.nrhs == nrhs)) {
            float ms = 0;
            if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) { tot += ms; n++; }
            ctx->prof_pool.push_back(r.a);
            ctx->prof_pool.push_back(r.b);
        } else {
            keep.push_back(r);
        }
    }
    ctx->prof.swap(keep);
    *total_ms = tot;
    *count = n;
    return TSM_OK;
}

size_t tsm_field_bytes(const tsm_ctx* ctx, int prec, int nrhs)
{
    if (!ctx || prec < 0 || prec > 2 || nrhs < 1) return 0;
    return field_bytes(prec, ctx->g.Vh, nrhs);
}

size_t tsm_workspace_bytes(const tsm_ctx* ctx, int max_nrhs, int prec)
{
    if (!ctx || max_nrhs < 1 || max_nrhs > TSM_MAX_NRHS || (prec != TSM_F64 && prec != TSM_F32)) return 0;
    return carve_workspace(const_cast<tsm_ctx*>(ctx), max_nrhs, prec, nullptr);
}

int tsm_set_workspace(tsm_ctx* ctx, void* dev_ptr, size_t bytes, int max_nrhs, int prec)
{
    if (!ctx) return TSM_EINVAL;
    if (!dev_ptr || max_nrhs < 1 || max_nrhs > TSM_MAX_NRHS || (prec != TSM_F64 && prec != TSM_F32)) return tsm_fail(ctx, TSM_EINVAL, "bad workspace arguments");
    if (((uintptr_t)dev_ptr & 255) != 0) return tsm_fail(ctx, TSM_EINVAL, "workspace must be 256-byte aligned");
    if (bytes < carve_workspace(ctx, max_nrhs, prec, nullptr)) return tsm_fail(ctx, TSM_EINVAL, "workspace too small");
    ctx->ws = (char*)dev_ptr;
    ctx->ws_bytes = bytes;
    ctx->max_nrhs = max_nrhs;
    ctx->ws_prec = prec;
    carve_workspace(ctx, max_nrhs, prec, ctx->ws);
    ctx->have_ws = true;
    ctx->have_gauge = false;
    ctx_drop_graphs(ctx);
    for (int s = 0; s < 2; s++) { ctx->slot_prec[s] = -1; ctx->slot_nrhs[s] = 0; }
    // the caller's buffer is uninitialised: start from the default operator set (16 local loops) with zeroed sums
    ctx->loops_ready = false;
    return tsm_loops_reset(ctx, 0);
}

int tsm_set_stream(tsm_ctx* ctx, void* cuda_stream)
{
    if (!ctx) return TSM_EINVAL;
    // the legacy default stream (NULL) cannot be captured into a CUDA graph: the library then uses its own
    // blocking stream, which keeps the legacy stream's ordering with the caller's default-stream work
    ctx->stream = cuda_stream ? (cudaStream_t)cuda_stream : ctx->own_stream;
    return TSM_OK;
}

int tsm_set_params(tsm_ctx* ctx, double kappa, double mu)
{
    if (!ctx) return TSM_EINVAL;
    if (!std::isfinite(kappa) || !std::isfinite(mu) || kappa == 0.0) return tsm_fail(ctx, TSM_EINVAL, "bad kappa/mu");
    ctx_drop_graphs(ctx);
    ctx->kappa = kappa;
    ctx->mu = mu;
    ctx->have_params = true;
    return TSM_OK;
}

int tsm_set_gauge(tsm_ctx* ctx, const double* host_links, int reconstruct, double* max_unitarity_dev)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if (!host_links || (reconstruct != 18 && reconstruct != 12)) return tsm_fail(ctx, TSM_EINVAL, "bad gauge arguments");
    ctx->have_gauge = false;
    if (reconstruct != ctx->recon) ctx_drop_graphs(ctx);   // other kernel variants; same pointers otherwise
    ctx->recon = reconstruct;
    const size_t bytes = (size_t)4 * ctx->g.V * 18 * sizeof(double);
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->staging, host_links, bytes, cudaMemcpyHostToDevice, ctx->stream));
    double* dev_max = (double*)ctx->cg->pq;   // scratch scalar
    rc = launch_gauge_pack(ctx, dev_max);
    if (rc) return rc;
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->host_small, dev_max, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    const double dev = ctx->host_small[0];
    if (max_unitarity_dev) *max_unitarity_dev = dev;
    if (!std::isfinite(dev)) return tsm_fail(ctx, TSM_EINVAL, "non-finite gauge links");
    if (reconstruct == 12 && dev > 1e-10) return tsm_fail(ctx, TSM_ENOTUNITARY, "links are not SU(3) to 1e-10; 12-real reconstruction refused");
    ctx->have_gauge = true;
    return TSM_OK;
}

int tsm_pack(tsm_ctx* ctx, int prec, int nrhs, const double* host_lex, void* dev_native)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if (!host_lex || !dev_native || nrhs < 1 || nrhs > ctx->max_nrhs || prec < 0 || prec > 2) return tsm_fail(ctx, TSM_EINVAL, "bad pack arguments");
    const size_t bytes = (size_t)nrhs * ctx->g.V * 24 * sizeof(double);
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->staging, host_lex, bytes, cudaMemcpyHostToDevice, ctx->stream));
    rc = launch_pack_spinor(ctx, prec, nrhs, (const double*)ctx->staging, dev_native);
    if (rc) return rc;
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return TSM_OK;
}

int tsm_unpack(tsm_ctx* ctx, int prec, int nrhs, const void* dev_native, double* host_lex)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if (!host_lex || !dev_native || nrhs < 1 || nrhs > ctx->max_nrhs || prec < 0 || prec > 2) return tsm_fail(ctx, TSM_EINVAL, "bad unpack arguments");
    rc = launch_unpack_spinor(ctx, prec, nrhs, dev_native, (double*)ctx->staging);
    if (rc) return rc;
    const size_t bytes = (size_t)nrhs * ctx->g.V * 24 * sizeof(double);
    TSM_CUDA(ctx, cudaMemcpyAsync(host_lex, ctx->staging, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    TSM_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return TSM_OK;
}

int tsm_noise(tsm_ctx* ctx, uint64_t seed, uint32_t source_id, int kind, double* host_out)
{
    int rc = ctx_enter(ctx, true, false, false);
    if (rc) return rc;
    if (!host_out || (kind != TSM_Z4 && kind != TSM_Z2)) return tsm_fail(ctx, TSM_EINVAL, "bad noise arguments");
    TSM_CUDA(ctx, cudaMemcpyAsync(ctx->ids_dev, &source_id, sizeof(uint32_t), cudaMemcpyHostToDevice, ctx->stream));
    const int np = ctx->ws_prec;   // the noise values (+-1, +-i) are exact in every precision
    rc = launch_noise(ctx, np, 1, seed, ctx->ids_dev, kind, ctx->vec[0]);
    if (rc) return rc;
    return tsm_unpack(ctx, np, 1, ctx->vec[0], host_out);
}

int tsm_dslash(tsm_ctx* ctx, int op, int prec, int nrhs, const void* dev_in, void* dev_out)
{
    int rc = ctx_enter(ctx, true, true, op != TSM_OP_D_EO && op != TSM_OP_D_OE);
    if (rc) return rc;
    if (!dev_in || !dev_out || dev_in == dev_out || nrhs < 1 || nrhs > ctx->max_nrhs || prec < 0 || prec > 2)
        return tsm_fail(ctx, TSM_EINVAL, "bad dslash arguments");
    if (prec == TSM_F64 && ctx->ws_prec != TSM_F64) return tsm_fail(ctx, TSM_ESTATE, "fp64 stencil on a low-precision-only workspace (tsm_set_workspace prec)");
    const double k = ctx->kappa, a = 2.0 * ctx->kappa * ctx->mu, n = 1.0 / (1.0 + a * a);
    const TwistCoef zero = {0, 0, 0, 0}, one = {1, 0, 1, 0};
    const TwistCoef R = {1, a, 1, -a}, Rinv = {n, -a * n, n, a * n}, Rb = {1, -a, 1, a}, Rbinv = {n, a * n, n, -a * n};
    const TwistCoef mk2 = {-k * k, 0, -k * k, 0}, mk = {-k, 0, -k, 0};
    switch (op) {
        case TSM_OP_D_EO: return launch_dslash(ctx, prec, 0, false, nrhs, dev_in, nullptr, dev_out, {zero, one}, 0);
        case TSM_OP_D_OE: return launch_dslash(ctx, prec, 1, false, nrhs, dev_in, nullptr, dev_out, {zero, one}, 0);
        case TSM_OP_MHAT:
            rc = launch_dslash(ctx, prec, 1, false, nrhs, dev_in, nullptr, ctx->vec[4], {zero, Rinv}, 0);
            if (rc) return rc;
            return launch_dslash(ctx, prec, 0, false, nrhs, ctx->vec[4], dev_in, dev_out, {R, mk2}, 0);
        case TSM_OP_MHAT_DAG:
            rc = launch_dslash(ctx, prec, 1, true, nrhs, dev_in, nullptr, ctx->vec[4], {zero, Rbinv}, 0);
            if (rc) return rc;
            return launch_dslash(ctx, prec, 0, true, nrhs, ctx->vec[4], dev_in, dev_out, {Rb, mk2}, 0);
        case TSM_OP_M_FULL: {
            const size_t fp = field_bytes(prec, ctx->g.Vh, nrhs);
            const char* in_e = (const char*)dev_in; const char* in_o = in_e + fp;
            char* out_e = (char*)dev_out; char* out_o = out_e + fp;
            rc = launch_dslash(ctx, prec, 0, false, nrhs, in_o, in_e, out_e, {R, mk}, 0);
            if (rc) return rc;
            return launch_dslash(ctx, prec, 1, false, nrhs, in_e, in_o, out_o, {R, mk}, 0);
        }
        default: return tsm_fail(ctx, TSM_EINVAL, "bad dslash op");
    }
}

}  // extern "C"
