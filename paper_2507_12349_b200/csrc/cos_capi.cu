// cos_capi.cu -- the extern "C" boundary declared in include/cos.h.
#include "../../include/cos.h"
#include "cos_compile.h"
#include "cos_kernels.cuh"

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

using namespace cosb;

namespace {

thread_local std::string g_err;

int fail(int code, const std::string& msg) { g_err = msg; return code; }
int cuda_fail(cudaError_t e, const char* what)
{
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? COS_ENOMEM : COS_ECUDA;
}

struct DeviceLayer { uint32_t* words = nullptr; uint32_t* mask_off = nullptr; uint32_t n_words = 0; };

// compile_dag reports structural limits with this prefix; everything else it returns is an out-of-memory condition
bool is_unsupported(const std::string& err) { return err.compare(0, 12, "unsupported:") == 0; }

}  // namespace

struct cos_handle_s {
    CompiledDag dag;
    bool on_device = false;
    int device = -1;
    std::vector<DeviceLayer> dl;
    size_t program_bytes = 0;
    double* ws = nullptr;                 // two ping-pong layer slabs
    size_t ws_bytes = 0;
    long long ws_limit = 64ll << 30;
    long long reserved_batch = 0;         // largest batch passed to cos_reserve (COS_INFO_RESERVED_BATCH)
    // launch shape and tuning (cos_set_tuning); nothing here is read from the environment
    int warps_per_cta = 8, ctas_per_sm = 1, n_sm = 148;
    int prefetch = 8;                     // L2 look-ahead distance in states
    int blocks_per_cta_cap = 0;           // 0: one block per staged table slot (64 .. 1024)
    int pdl = 1;                          // programmatic dependent launch between layers
    int host_slices = 8;                  // cos_eval_host: at most this many output slices (1: no second stream)
    long long tiles_per_chunk = 0;        // 0: as many batch tiles per workspace chunk as the limit allows
    bool fused_ok = false;                // small DAG: every layer can run in one launch (cos_fused_kernel)
    bool fused = false;                   // ... and does
    FusedLayer* fused_layers = nullptr;   // device array
    long long n_launches = 0;
    // profiling (cos_set_profiling): events[k*(NL+1) + l] brackets layer l of the k-th profiled chunk
    bool profiling = false;
    std::vector<cudaEvent_t> events;
    size_t events_used = 0;
    long long profiled_evals = 0;
    // staging of cos_eval_host
    int* st_sites = nullptr; double* st_tau = nullptr; double* st_G = nullptr; double* st_out = nullptr;
    long long st_batch = 0;
    cudaStream_t copy_stream = nullptr;   // D2H of finished output slices (cos_eval_host)
    cudaEvent_t copy_events[8] = {};
};

struct cos_tab_s {
    double* T = nullptr;
    int device = -1;
    int lattice = 0, L = 0, nsub = 1, n_blocks = 1, n_tau = 0;
    double beta = 0.0;
};

extern "C" {

const char* cos_last_error(void) { return g_err.c_str(); }

static int build_impl(int n, int n_flavors, int lattice, const double* shifts, int readout_envelope,
                      unsigned int order_mask, int flags, cos_handle* out);

int cos_build_ex(int n, int n_flavors, int lattice, const double* shifts, int readout_envelope, int flags,
                 cos_handle* out)
{
    return build_impl(n, n_flavors, lattice, shifts, readout_envelope, 0u, flags, out);
}

int cos_build_orders(int n, int n_flavors, int lattice, const double* shifts, unsigned int order_mask, int flags,
                     cos_handle* out)
{
    if (n >= 1 && n <= COS_MAX_N && (order_mask & ((2u << n) - 2u)) == 0u) {
        if (out) *out = nullptr;
        return fail(COS_EINVAL, "cos_build_orders: order_mask selects no order in [1, n]");
    }
    return build_impl(n, n_flavors, lattice, shifts, n, order_mask & ((2u << n) - 2u), flags, out);
}

static int build_impl(int n, int n_flavors, int lattice, const double* shifts, int readout_envelope,
                      unsigned int order_mask, int flags, cos_handle* out)
{
    if (!out) return fail(COS_EINVAL, "cos_build: out is NULL");
    *out = nullptr;
    if (n < 1 || n > COS_MAX_N) return fail(COS_EINVAL, "cos_build: n must be in [1, 12]");
    if (n_flavors < 1) return fail(COS_EINVAL, "cos_build: n_flavors must be >= 1");
    if (lattice != COS_LATTICE_SQUARE && lattice != COS_LATTICE_HONEYCOMB)
        return fail(COS_EINVAL, "cos_build: unknown lattice");
    if (readout_envelope != 0 && readout_envelope != n)
        return fail(COS_EINVAL, "cos_build: readout_envelope must be 0 or n");
    const bool uniform_shift = (flags & COS_BUILD_UNIFORM_SHIFT) != 0;
    if (uniform_shift && !shifts) return fail(COS_EINVAL, "cos_build: COS_BUILD_UNIFORM_SHIFT needs shifts[0]");
    if (shifts && !uniform_shift && n_flavors > COS_MAX_COLOURS)
        return fail(COS_EUNSUPPORTED, "cos_build: SB-CoS supports at most 4 flavours");
    const int nsub = lattice == COS_LATTICE_HONEYCOMB ? 2 : 1;
    if (n * nsub > 24) return fail(COS_EUNSUPPORTED, "cos_build: n * n_sub must be <= 24");

    cos_handle_s* h = new (std::nothrow) cos_handle_s();
    if (!h) return fail(COS_ENOMEM, "cos_build: out of host memory");
    std::string err = compile_dag(n, n_flavors, nsub, shifts, uniform_shift, readout_envelope == n, order_mask, h->dag);
    if (!err.empty()) {
        delete h;
        return fail(is_unsupported(err) ? COS_EUNSUPPORTED : COS_ENOMEM, "cos_build: " + err);
    }

    const CompiledDag& D = h->dag;
    const size_t smem = layer_smem_bytes(D.n_blocks * D.d * D.d, D.nc, D.d, D.has_shift);
    if (smem > LAYER_SMEM_MAX) {
        delete h;
        return fail(COS_EUNSUPPORTED, "cos_build: propagator tile does not fit the 226 KB of shared memory a CTA can use for it (227 KB per SM minus 1 KB of bookkeeping)");
    }

    if (!(flags & COS_BUILD_HOST_ONLY)) {
        int ndev = 0;
        cudaError_t e = cudaGetDeviceCount(&ndev);
        if (e != cudaSuccess || ndev == 0) {
            delete h;
            return fail(COS_ECUDA, "cos_build: no CUDA device (there is no CPU fallback; use COS_BUILD_HOST_ONLY to inspect the DAG)");
        }
        cudaGetDevice(&h->device);
        e = configure_layer_kernels();
        if (e != cudaSuccess) { delete h; return cuda_fail(e, "cos_build: cudaFuncSetAttribute"); }
        // launch shape: the CTA size that keeps the most warps resident per SM
        e = pick_layer_shape((int)D.max_L, D.nc, D.d, D.n_blocks * D.d * D.d, D.has_shift, &h->warps_per_cta, &h->ctas_per_sm);
        if (e != cudaSuccess) { delete h; return cuda_fail(e, "cos_build: occupancy query"); }
        cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device);
        h->dl.resize(D.layers.size());
        for (size_t l = 0; l < D.layers.size(); ++l) {
            const LayerProgram& P = D.layers[l];
            const size_t wb = P.words.size() * sizeof(uint32_t), mb = P.mask_off.size() * sizeof(uint32_t);
            if (wb == 0) continue;
            h->dl[l].n_words = (uint32_t)P.words.size();
            e = cudaMalloc(&h->dl[l].words, wb);
            if (e == cudaSuccess) e = cudaMalloc(&h->dl[l].mask_off, mb);
            if (e == cudaSuccess) e = cudaMemcpy(h->dl[l].words, P.words.data(), wb, cudaMemcpyHostToDevice);
            if (e == cudaSuccess) e = cudaMemcpy(h->dl[l].mask_off, P.mask_off.data(), mb, cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { cos_free(h); return cuda_fail(e, "cos_build: uploading the layer program"); }
            h->program_bytes += wb + mb;
        }
        // small DAGs (orders n <= 6) are launch-latency bound: walk all layers in one kernel
        bool small = D.n_states <= 16384 && D.max_L <= 12;
        for (const auto& P : D.layers) small = small && P.n_masks <= 2048;
        if (small) {
            std::vector<FusedLayer> fl(D.layers.size());
            for (size_t l = 0; l < D.layers.size(); ++l) {
                fl[l].words = h->dl[l].words; fl[l].mask_off = h->dl[l].mask_off;
                fl[l].n_masks = D.layers[l].n_masks; fl[l].n_states = D.layers[l].n_states; fl[l].n_words = h->dl[l].n_words;
            }
            e = cudaMalloc(&h->fused_layers, fl.size() * sizeof(FusedLayer));
            if (e == cudaSuccess) e = cudaMemcpy(h->fused_layers, fl.data(), fl.size() * sizeof(FusedLayer), cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { cos_free(h); return cuda_fail(e, "cos_build: fused-path setup"); }
            h->fused_ok = true;
            h->fused = !(flags & COS_BUILD_NO_FUSED);
        }
        h->on_device = true;
        // the host copy of the program is no longer needed
        for (auto& P : h->dag.layers) { std::vector<uint32_t>().swap(P.words); std::vector<uint32_t>().swap(P.mask_off); }
    } else {
        for (const auto& P : D.layers) h->program_bytes += (P.words.size() + P.mask_off.size()) * sizeof(uint32_t);
    }
    *out = h;
    return COS_OK;
}

int cos_build(int n, int n_flavors, int lattice, const double* shifts, int readout_envelope, cos_handle* out)
{
    return cos_build_ex(n, n_flavors, lattice, shifts, readout_envelope, 0, out);
}

void cos_free(cos_handle h)
{
    if (!h) return;
    for (auto& l : h->dl) { if (l.words) cudaFree(l.words); if (l.mask_off) cudaFree(l.mask_off); }
    if (h->ws) cudaFree(h->ws);
    if (h->fused_layers) cudaFree(h->fused_layers);
    for (cudaEvent_t e : h->events) cudaEventDestroy(e);
    if (h->st_sites) cudaFree(h->st_sites);
    if (h->st_tau) cudaFree(h->st_tau);
    if (h->st_G) cudaFree(h->st_G);
    if (h->st_out) cudaFree(h->st_out);
    if (h->copy_stream) {
        cudaStreamDestroy(h->copy_stream);
        for (cudaEvent_t ev : h->copy_events) if (ev) cudaEventDestroy(ev);
    }
    delete h;
}

int cos_set_workspace_limit(cos_handle h, long long bytes)
{
    if (!h || bytes <= 0) return fail(COS_EINVAL, "cos_set_workspace_limit: bad argument");
    h->ws_limit = bytes;
    return COS_OK;
}

// The handle's device must be the current one: its program, workspace and the caller's pointers live there.
static int check_device(cos_handle h, const char* who)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, who);
    if (dev != h->device)
        return fail(COS_EINVAL, std::string(who) + ": the current CUDA device is not the one the handle was built on");
    return COS_OK;
}

// Batch tiles per workspace chunk for a batch of `batch` configurations, and the bytes that chunk needs.
static long long chunk_tiles(cos_handle h, long long batch, size_t* bytes)
{
    const CompiledDag& D = h->dag;
    const long long tiles_total = (batch + TILE - 1) / TILE;
    const size_t tile_bytes = (size_t)D.max_layer_states * TILE * sizeof(double) * 2;
    long long tiles_chunk = (long long)((size_t)h->ws_limit / tile_bytes);
    if (tiles_chunk < 1) tiles_chunk = 1;
    if (tiles_chunk > tiles_total) tiles_chunk = tiles_total;
    if (h->tiles_per_chunk > 0 && tiles_chunk > h->tiles_per_chunk) tiles_chunk = h->tiles_per_chunk;
    *bytes = tile_bytes * (size_t)tiles_chunk;
    return tiles_chunk;
}

// stream: the stream the caller is about to enqueue on, or nullptr when there is none (cos_reserve).  Growing the
// workspace is a cudaFree + cudaMalloc: never while that stream is being captured -- it would break the capture, and a
// graph captured earlier holds the old pointer.
static int grow_workspace(cos_handle h, size_t need, const char* who, cudaStream_t stream, bool have_stream)
{
    if (need <= h->ws_bytes) return COS_OK;
    if (have_stream) {
        cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
        cudaError_t eq = cudaStreamIsCapturing(stream, &st);
        if (eq != cudaSuccess) return cuda_fail(eq, who);
        if (st != cudaStreamCaptureStatusNone)
            return fail(COS_EINVAL, std::string(who) + ": the workspace would have to grow (" + std::to_string(h->ws_bytes) +
                        " -> " + std::to_string(need) + " bytes) while the stream is being captured; call cos_reserve for this "
                        "batch before the capture begins");
    }
    if (h->ws) { cudaFree(h->ws); h->ws = nullptr; h->ws_bytes = 0; }
    cudaError_t e = cudaMalloc(&h->ws, need);
    if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e, who); }
    h->ws_bytes = need;
    return COS_OK;
}

int cos_reserve(cos_handle h, long long batch)
{
    if (!h || batch < 0) return fail(COS_EINVAL, "cos_reserve: bad argument");
    if (!h->on_device) return fail(COS_ECUDA, "cos_reserve: handle was built host-only (no CPU fallback)");
    int rc = check_device(h, "cos_reserve");
    if (rc != COS_OK || batch == 0) return rc;
    size_t need = 0;
    chunk_tiles(h, batch, &need);
    rc = grow_workspace(h, need, "cos_reserve: workspace allocation", nullptr, false);
    if (rc == COS_OK && batch > h->reserved_batch) h->reserved_batch = batch;
    return rc;
}

int cos_set_tuning(cos_handle h, int what, long long value)
{
    if (!h) return fail(COS_EINVAL, "cos_set_tuning: handle is NULL");
    switch (what) {
        case COS_TUNE_PREFETCH:
            if (value < 0 || value > 4096) return fail(COS_EINVAL, "cos_set_tuning: prefetch distance must be in [0, 4096]");
            h->prefetch = (int)value; break;
        case COS_TUNE_WARPS_PER_CTA:
            if (value < 1 || value > 24) return fail(COS_EINVAL, "cos_set_tuning: warps per CTA must be in [1, 24]");
            if (h->on_device) {       // resident CTAs per SM for the new shape (sizes the grid waves)
                const int rcd = check_device(h, "cos_set_tuning");     // the occupancy query is about the handle's device
                if (rcd != COS_OK) return rcd;
                const CompiledDag& D = h->dag;
                int c = 0;
                if (layer_ctas_per_sm((int)D.max_L, D.nc, D.d, D.n_blocks * D.d * D.d, D.has_shift, (int)value, &c) != cudaSuccess || c < 1) {
                    cudaGetLastError();
                    return fail(COS_EINVAL, "cos_set_tuning: this CTA size does not fit the handle's kernel");
                }
                h->ctas_per_sm = c;
            }
            h->warps_per_cta = (int)value;
            break;
        case COS_TUNE_BLOCKS_PER_CTA_CAP:
            if (value < 0 || value > 65535) return fail(COS_EINVAL, "cos_set_tuning: blocks-per-CTA cap must be in [0, 65535]");
            h->blocks_per_cta_cap = (int)value; break;
        case COS_TUNE_PDL: h->pdl = value != 0; break;
        case COS_TUNE_FUSED: h->fused = h->fused_ok && value != 0; break;
        case COS_TUNE_HOST_SLICES:
            if (value < 1 || value > 8) return fail(COS_EINVAL, "cos_set_tuning: host slices must be in [1, 8]");
            h->host_slices = (int)value; break;
        case COS_TUNE_TILES_PER_CHUNK:
            if (value < 0) return fail(COS_EINVAL, "cos_set_tuning: tiles per chunk must be >= 0");
            h->tiles_per_chunk = value; break;
        default: return fail(COS_EINVAL, "cos_set_tuning: unknown parameter");
    }
    return COS_OK;
}

// Layers + readouts for the batch tiles [tile_begin, tile_end) of a batch of `batch` configurations (G_dev / out_dev are
// the whole-batch arrays).  clear: zero-fill the output rows of a partial readout set first (whole batch).
static int eval_range(cos_handle h, const double* G_dev, long long batch, double* out_dev, long long tile_begin,
                      long long tile_end, bool clear, cudaStream_t stream)
{
    const CompiledDag& D = h->dag;
    const int NL = (int)D.layers.size();

    // ---- batch chunking against the workspace budget: two slabs of max_layer_states x 32 doubles per tile
    size_t need = 0;
    const long long tiles_chunk = chunk_tiles(h, batch, &need);
    // (cos_reserve hoists this allocation out of the call; growing here synchronises the device)
    int rc = grow_workspace(h, need, "cos_eval: workspace allocation", stream, true);
    if (rc != COS_OK) return rc;
    double* slab[2] = {h->ws, h->ws + (size_t)D.max_layer_states * TILE * (size_t)tiles_chunk};
#ifdef COS_CHECK_BOUNDS
    // self-check build: the slabs start as NaN, so a state that is read before it was written shows in the outputs
    if (cudaMemsetAsync(h->ws, 0xFF, need, stream) != cudaSuccess) cudaGetLastError();
#endif

    if (clear && D.all_subsets && D.order_mask != (((2u << D.n) - 1u) & ~1u)) {     // partial readout set: other rows are zeros
        cudaError_t e = cudaMemsetAsync(out_dev, 0, (size_t)D.n_out * (size_t)batch * sizeof(double), stream);
        if (e != cudaSuccess) return cuda_fail(e, "cos_eval: clearing the output");
    }
    const int n_slots = D.n_blocks * D.d * D.d;
    for (long long t0 = tile_begin; t0 < tile_end; t0 += tiles_chunk) {
        const uint32_t tiles = (uint32_t)((tile_end - t0 < tiles_chunk) ? (tile_end - t0) : tiles_chunk);
        if (h->fused && !h->profiling) {
            FusedArgs f;
            f.layers = h->fused_layers; f.n_layers = NL; f.ws = h->ws; f.S_max = D.max_layer_states;
            f.G = G_dev; f.batch = batch; f.b0 = t0 * TILE; f.out = out_dev; f.d = D.d; f.n_slots = n_slots;
            f.neg_kappa = -D.kappa; f.n_out = (uint32_t)D.n_out;
            for (int c = 0; c < 4; ++c) f.sigma[c] = D.sigma[c];
            cudaError_t ef = launch_fused(f, (int)D.max_L, D.nc, D.has_shift, tiles, 8, stream);
            if (ef != cudaSuccess) return cuda_fail(ef, "cos_eval: fused launch");
            ++h->n_launches;
            continue;
        }
        cudaError_t e = launch_fill_ones(slab[0], (size_t)D.layers[0].n_states * TILE * tiles, stream);
        if (e != cudaSuccess) return cuda_fail(e, "cos_eval: fill launch");
        ++h->n_launches;
        cudaEvent_t* ev = nullptr;
        if (h->profiling) {
            const size_t need_ev = h->events_used + (size_t)NL + 1;
            while (h->events.size() < need_ev) {
                cudaEvent_t x;
                e = cudaEventCreate(&x);
                if (e != cudaSuccess) return cuda_fail(e, "cos_eval: cudaEventCreate");
                h->events.push_back(x);
            }
            ev = h->events.data() + h->events_used;
            h->events_used = need_ev;
            cudaEventRecord(ev[0], stream);
        }
        for (int l = 0; l < NL; ++l) {
            const LayerProgram& P = D.layers[l];
            LayerArgs a;
            a.words = h->dl[l].words; a.mask_off = h->dl[l].mask_off;
            a.n_masks = P.n_masks; a.n_words = h->dl[l].n_words; a.n_out = (uint32_t)D.n_out;
            {   // blocks per CTA: amortise the table staging but keep >= 4 waves of CTAs on the GPU
                const long long resident = (long long)h->n_sm * h->ctas_per_sm;
                long long mpc = (long long)P.n_masks * tiles / (resident * 4);
                // staging the table costs one 256-byte line per slot and CTA; a block moves ~30 lines each way:
                // about one block per staged slot keeps the staging share at a few percent
                long long cap = n_slots + (D.has_shift ? D.nc * D.d : 0);
                if (cap < 64) cap = 64;
                if (cap > 1024) cap = 1024;
                if (h->blocks_per_cta_cap > 0) cap = h->blocks_per_cta_cap;
                if (mpc > cap) mpc = cap;
                // small layers (few blocks x few tiles): one wave of CTAs, so that every block finds a warp at once
                // (a block is walked by ONE warp, latency-bound), but never more than two blocks per warp
                long long floor_ = (P.n_masks * (long long)tiles + resident - 1) / resident;
                if (floor_ > 2 * h->warps_per_cta) floor_ = 2 * h->warps_per_cta;
                if (floor_ < 1) floor_ = 1;
                if (mpc < floor_) mpc = floor_;
                while ((P.n_masks + mpc - 1) / mpc > 65535) mpc *= 2;
                a.masks_per_cta = (uint32_t)mpc;
            }
            a.prefetch = h->prefetch;
            a.pdl = (h->pdl && l > 0 && !h->profiling) ? 1 : 0;   // per-layer events need serialised layers
            a.X = slab[l & 1]; a.Y = slab[(l + 1) & 1];
            a.S_src = P.n_states; a.S_dst = (l + 1 < NL) ? D.layers[l + 1].n_states : 0;
            a.G = G_dev; a.batch = batch; a.b0 = t0 * TILE; a.out = out_dev;
            a.d = D.d; a.n_slots = n_slots;
            a.neg_kappa = -D.kappa;
            for (int c = 0; c < 4; ++c) a.shift[c] = (l == 0 ? -2.0 : -1.0) * D.sigma[c];
            e = launch_layer(a, (int)D.max_L, D.nc, D.has_shift, tiles, h->warps_per_cta, stream);
            if (e != cudaSuccess) return cuda_fail(e, "cos_eval: layer launch");
            if (P.n_masks) ++h->n_launches;
            if (ev) cudaEventRecord(ev[l + 1], stream);
        }
    }
    return COS_OK;
}

int cos_eval(cos_handle h, const double* G_dev, long long batch, double* out_dev, cos_stream stream_)
{
    if (!h) return fail(COS_EINVAL, "cos_eval: handle is NULL");
    if (batch < 0) return fail(COS_EINVAL, "cos_eval: negative batch");
    if (batch == 0) return COS_OK;
    if (!G_dev || !out_dev) return fail(COS_EINVAL, "cos_eval: NULL device pointer");
    if (!h->on_device) return fail(COS_ECUDA, "cos_eval: handle was built host-only / without a CUDA device (no CPU fallback)");
    int rc = check_device(h, "cos_eval");
    if (rc != COS_OK) return rc;
    if (h->profiling) ++h->profiled_evals;
    return eval_range(h, G_dev, batch, out_dev, 0, (batch + TILE - 1) / TILE, true, (cudaStream_t)stream_);
}

int cos_set_profiling(cos_handle h, int on)
{
    if (!h) return fail(COS_EINVAL, "cos_set_profiling: handle is NULL");
    h->profiling = on != 0;
    return COS_OK;
}

int cos_get_layer_times(cos_handle h, int n_layers, double* ms, long long* n_evals)
{
    if (!h || !ms || n_layers < 0) return fail(COS_EINVAL, "cos_get_layer_times: bad argument");
    const int NL = (int)h->dag.layers.size();
    const size_t per = (size_t)NL + 1;
    for (size_t k = 0; k + per <= h->events_used; k += per) {
        cudaError_t e = cudaEventSynchronize(h->events[k + NL]);
        if (e != cudaSuccess) return cuda_fail(e, "cos_get_layer_times: cudaEventSynchronize");
        for (int l = 0; l < NL && l < n_layers; ++l) {
            float t = 0.f;
            e = cudaEventElapsedTime(&t, h->events[k + l], h->events[k + l + 1]);
            if (e != cudaSuccess) return cuda_fail(e, "cos_get_layer_times: cudaEventElapsedTime");
            ms[l] += (double)t;
        }
    }
    if (n_evals) *n_evals = h->profiled_evals;
    h->events_used = 0;
    h->profiled_evals = 0;
    return COS_OK;
}

int cos_eval_host(cos_handle h, cos_tab tab, const int* sites_host, const double* tau_host, long long batch,
                  double* out_host, cos_stream stream_)
{
    if (!h || !tab) return fail(COS_EINVAL, "cos_eval_host: NULL handle");
    if (batch < 0) return fail(COS_EINVAL, "cos_eval_host: negative batch");
    if (batch == 0) return COS_OK;
    if (!sites_host || !tau_host || !out_host) return fail(COS_EINVAL, "cos_eval_host: NULL host pointer");
    if (!h->on_device) return fail(COS_ECUDA, "cos_eval_host: handle was built host-only (no CPU fallback)");
    {
        const int rcd = check_device(h, "cos_eval_host");
        if (rcd != COS_OK) return rcd;
    }
    const CompiledDag& D = h->dag;
    if (tab->n_blocks != D.n_blocks || tab->nsub != D.nsub)
        return fail(COS_EINVAL, "cos_eval_host: table blocks / lattice do not match the handle");
    cudaStream_t stream = (cudaStream_t)stream_;
    const size_t B = (size_t)batch, n = (size_t)D.n;
    const size_t b_sites = n * 2 * B * sizeof(int), b_tau = n * B * sizeof(double);
    const size_t b_G = (size_t)D.n_blocks * D.d * D.d * B * sizeof(double), b_out = (size_t)D.n_out * B * sizeof(double);
    if (batch > h->st_batch) {
        if (h->st_sites) cudaFree(h->st_sites);
        if (h->st_tau) cudaFree(h->st_tau);
        if (h->st_G) cudaFree(h->st_G);
        if (h->st_out) cudaFree(h->st_out);
        h->st_sites = nullptr; h->st_tau = nullptr; h->st_G = nullptr; h->st_out = nullptr; h->st_batch = 0;
        cudaError_t e = cudaMalloc(&h->st_sites, b_sites);
        if (e == cudaSuccess) e = cudaMalloc(&h->st_tau, b_tau);
        if (e == cudaSuccess) e = cudaMalloc(&h->st_G, b_G);
        if (e == cudaSuccess) e = cudaMalloc(&h->st_out, b_out);
        if (e != cudaSuccess) { cudaGetLastError(); return cuda_fail(e, "cos_eval_host: staging allocation"); }
        h->st_batch = batch;
    }
    cudaError_t e = cudaMemcpyAsync(h->st_sites, sites_host, b_sites, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h->st_tau, tau_host, b_tau, cudaMemcpyHostToDevice, stream);
    if (e != cudaSuccess) return cuda_fail(e, "cos_eval_host: host-to-device copy");
    int rc = cos_tabulate(tab, D.n, h->st_sites, h->st_tau, batch, h->st_G, stream_);
    if (rc != COS_OK) return rc;
    ++h->n_launches;
    if (h->profiling) ++h->profiled_evals;
    // Large outputs (all-subset readouts): walk the batch in up to 8 slices and copy the output columns of slice i
    // back on a second stream while slice i+1 is evaluated (one strided 2-D copy per slice).
    const long long tiles_total = (batch + TILE - 1) / TILE;
    long long n_slices = (long long)(b_out >> 23);                  // ~8 MiB of output per slice
    if (n_slices > h->host_slices) n_slices = h->host_slices;
    if (n_slices > tiles_total) n_slices = tiles_total;
    if (n_slices <= 1) {
        rc = eval_range(h, h->st_G, batch, h->st_out, 0, tiles_total, true, stream);
        if (rc != COS_OK) return rc;
        e = cudaMemcpyAsync(out_host, h->st_out, b_out, cudaMemcpyDeviceToHost, stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) return cuda_fail(e, "cos_eval_host: device-to-host copy");
        return COS_OK;
    }
    if (!h->copy_stream) {
        e = cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking);
        for (int i = 0; i < 8 && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&h->copy_events[i], cudaEventDisableTiming);
        if (e != cudaSuccess) return cuda_fail(e, "cos_eval_host: copy stream");
    }
    for (long long i = 0; i < n_slices; ++i) {
        const long long t_a = tiles_total * i / n_slices, t_b = tiles_total * (i + 1) / n_slices;
        rc = eval_range(h, h->st_G, batch, h->st_out, t_a, t_b, i == 0, stream);
        if (rc != COS_OK) {                       // no copy into out_host may still be in flight when the caller sees the error
            const std::string msg = g_err;
            cudaStreamSynchronize(h->copy_stream);
            cudaStreamSynchronize(stream);
            g_err = msg;
            return rc;
        }
        const size_t c0 = (size_t)t_a * TILE, c1 = (size_t)(t_b * TILE < batch ? t_b * TILE : batch);
        e = cudaEventRecord(h->copy_events[i], stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(h->copy_stream, h->copy_events[i], 0);
        if (e == cudaSuccess)
            e = cudaMemcpy2DAsync(out_host + c0, B * sizeof(double), h->st_out + c0, B * sizeof(double),
                                  (c1 - c0) * sizeof(double), (size_t)D.n_out, cudaMemcpyDeviceToHost, h->copy_stream);
        if (e != cudaSuccess) {
            cudaStreamSynchronize(h->copy_stream);
            cudaStreamSynchronize(stream);
            return cuda_fail(e, "cos_eval_host: pipelined device-to-host copy");
        }
    }
    e = cudaStreamSynchronize(h->copy_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return cuda_fail(e, "cos_eval_host: device-to-host copy");
    return COS_OK;
}

int cos_info(cos_handle h, int what, long long* value)
{
    if (!h || !value) return fail(COS_EINVAL, "cos_info: NULL argument");
    const CompiledDag& D = h->dag;
    const int NL = (int)D.layers.size();
    if (what >= COS_INFO_LAYER_STATES && what < COS_INFO_LAYER_STATES + NL) { *value = D.layers[what - COS_INFO_LAYER_STATES].n_states; return COS_OK; }
    if (what >= COS_INFO_LAYER_EDGES && what < COS_INFO_LAYER_EDGES + NL) {
        const LayerProgram& P = D.layers[what - COS_INFO_LAYER_EDGES];
        *value = (long long)(P.e1 + P.e2 + P.e3 + P.e4 + P.readout_edges); return COS_OK;
    }
    if (what >= COS_INFO_LAYER_MASKS && what < COS_INFO_LAYER_MASKS + NL) { *value = D.layers[what - COS_INFO_LAYER_MASKS].n_masks; return COS_OK; }
    switch (what) {
        case COS_INFO_N_LAYERS: *value = NL; break;
        case COS_INFO_N_STATES: *value = (long long)D.n_states; break;
        case COS_INFO_N_EDGES: *value = (long long)D.n_edges; break;
        case COS_INFO_N_READOUT_EDGES: *value = (long long)D.n_readout_edges; break;
        case COS_INFO_N_OUT: *value = D.n_out; break;
        case COS_INFO_MAX_LAYER_STATES: *value = D.max_layer_states; break;
        case COS_INFO_N_MASKS: *value = (long long)D.n_masks; break;
        case COS_INFO_N_ROWS: *value = (long long)D.n_rows; break;
        case COS_INFO_N_FMA: *value = (long long)D.n_fma; break;
        case COS_INFO_PROGRAM_BYTES: *value = (long long)h->program_bytes; break;
        case COS_INFO_D: *value = D.d; break;
        case COS_INFO_N_BLOCKS: *value = D.n_blocks; break;
        case COS_INFO_N_STATES_UNPRUNED: *value = (long long)D.n_states_unpruned; break;
        case COS_INFO_WORKSPACE_BYTES: *value = (long long)h->ws_bytes; break;
        case COS_INFO_N_LAUNCHES: *value = h->n_launches; break;
        case COS_INFO_ORDER_MASK: *value = (long long)D.order_mask; break;
        case COS_INFO_RESERVED_BATCH: *value = h->reserved_batch; break;
        case COS_INFO_DEVICE: *value = h->device; break;
        case COS_INFO_FUSED: *value = h->fused ? 1 : 0; break;
        default: return fail(COS_EINVAL, "cos_info: unknown query");
    }
    return COS_OK;
}

int cos_tab_build(int lattice, int L, int n_blocks, double beta, int n_tau, const double* table_host, cos_tab* out)
{
    if (!out) return fail(COS_EINVAL, "cos_tab_build: out is NULL");
    *out = nullptr;
    if (!table_host || L < 1 || n_blocks < 1 || n_tau < 2 || !(beta > 0.0) ||
        (lattice != COS_LATTICE_SQUARE && lattice != COS_LATTICE_HONEYCOMB))
        return fail(COS_EINVAL, "cos_tab_build: bad argument");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(COS_ECUDA, "cos_tab_build: no CUDA device");
    cos_tab_s* t = new (std::nothrow) cos_tab_s();
    if (!t) return fail(COS_ENOMEM, "cos_tab_build: out of host memory");
    cudaGetDevice(&t->device);
    t->lattice = lattice; t->L = L; t->nsub = lattice == COS_LATTICE_HONEYCOMB ? 2 : 1;
    t->n_blocks = n_blocks; t->n_tau = n_tau; t->beta = beta;
    const size_t bytes = (size_t)n_blocks * t->nsub * t->nsub * L * L * n_tau * sizeof(double);
    cudaError_t e = cudaMalloc(&t->T, bytes);
    if (e == cudaSuccess) e = cudaMemcpy(t->T, table_host, bytes, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { if (t->T) cudaFree(t->T); delete t; cudaGetLastError(); return cuda_fail(e, "cos_tab_build"); }
    *out = t;
    return COS_OK;
}

int cos_tabulate(cos_tab tab, int n, const int* sites_dev, const double* tau_dev, long long batch, double* G_dev,
                 cos_stream stream)
{
    if (!tab || n < 1 || n > COS_MAX_N || batch < 0) return fail(COS_EINVAL, "cos_tabulate: bad argument");
    if (batch == 0) return COS_OK;
    if (!sites_dev || !tau_dev || !G_dev) return fail(COS_EINVAL, "cos_tabulate: NULL device pointer");
    {
        int dev = -1;
        if (cudaGetDevice(&dev) != cudaSuccess || dev != tab->device)
            return fail(COS_EINVAL, "cos_tabulate: the current CUDA device is not the one the table was built on");
    }
    TabArgs a;
    a.T = tab->T; a.L = tab->L; a.nsub = tab->nsub; a.n_blocks = tab->n_blocks; a.n_tau = tab->n_tau; a.beta = tab->beta;
    a.n = n; a.sites = sites_dev; a.tau = tau_dev; a.batch = batch; a.G = G_dev;
    cudaError_t e = launch_tabulate(a, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "cos_tabulate: launch");
    return COS_OK;
}

void cos_tab_free(cos_tab tab)
{
    if (!tab) return;
    if (tab->T) cudaFree(tab->T);
    delete tab;
}

int cos_flux_weights(int n, unsigned int order_mask, const double* lambda_host, const double* C_dev,
                     const double* Q_dev, long long batch, double* W_dev, double* Phi_dev, cos_stream stream)
{
    if (n < 1 || n > COS_MAX_N || batch < 0) return fail(COS_EINVAL, "cos_flux_weights: bad argument");
    if (batch == 0) return COS_OK;
    if (!lambda_host || !C_dev || !W_dev) return fail(COS_EINVAL, "cos_flux_weights: NULL pointer");
    FluxArgs a;
    a.n = n;
    a.order_mask = order_mask ? (order_mask & ((2u << n) - 2u)) : ((2u << n) - 2u);
    if (a.order_mask == 0u) return fail(COS_EINVAL, "cos_flux_weights: order_mask selects no order in [1, n]");
    double b = 1.0;                                   // binom(n, k), exact in fp64 for n <= 12
    for (int k = 0; k <= 12; ++k) {
        a.lambda[k] = (k >= 1 && k <= n) ? lambda_host[k] : 0.0;
        a.binom[k] = (k <= n) ? b : 1.0;
        if (k < n) b = b * (double)(n - k) / (double)(k + 1);
    }
    a.C = C_dev; a.Q = Q_dev; a.W = W_dev; a.Phi = Phi_dev; a.batch = batch;
    cudaError_t e = launch_flux(a, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "cos_flux_weights: launch");
    return COS_OK;
}

long long cos_det_workspace_bytes(int n, int n_blocks, int precision, long long batch)
{
    if (n < 1 || n > COS_MAX_N || n_blocks < 1 || n_blocks > 3 || batch < 0 || (precision != COS_DET_FP64 && precision != COS_DET_DD))
        return -1;
    const long long elem = precision == COS_DET_DD ? 16 : 8;
    return elem * (n_blocks + 2) * (1ll << n) * batch + (long long)sizeof(uint32_t) * (1ll << n);
}

int cos_det_eval(int n, int n_flavors, int n_blocks, int lattice, const double* shifts, int precision,
                 const double* G_dev, long long batch, double* out_dev, void* work_dev, long long work_bytes,
                 cos_stream stream)
{
    if (n < 1 || n > COS_MAX_N || batch < 0) return fail(COS_EINVAL, "cos_det_eval: bad n or batch");
    if (lattice != COS_LATTICE_SQUARE && lattice != COS_LATTICE_HONEYCOMB) return fail(COS_EINVAL, "cos_det_eval: bad lattice");
    if (precision != COS_DET_FP64 && precision != COS_DET_DD) return fail(COS_EINVAL, "cos_det_eval: bad precision");
    if (n_flavors != 2 && n_flavors != 3)
        return fail(COS_EUNSUPPORTED, "cos_det_eval: the local tensor of Eq. 35 is implemented for 2 or 3 flavours");
    if (n_blocks != 1 && n_blocks != n_flavors) return fail(COS_EINVAL, "cos_det_eval: n_blocks must be 1 or n_flavors");
    if (batch == 0) return COS_OK;
    if (!G_dev || !out_dev || !work_dev) return fail(COS_EINVAL, "cos_det_eval: NULL pointer");
    if (((size_t)work_dev & 15u) != 0) return fail(COS_EINVAL, "cos_det_eval: work_dev must be 16-byte aligned");
    if (work_bytes < cos_det_workspace_bytes(n, n_blocks, precision, batch))
        return fail(COS_EINVAL, "cos_det_eval: workspace smaller than cos_det_workspace_bytes");
    if (batch > 0x7fffffffll || (((1ll << n) - 1) * ((batch + 31) / 32)) > 0x7fffffffll)
        return fail(COS_EUNSUPPORTED, "cos_det_eval: (2^n - 1) * ceil(batch / 32) exceeds the grid limit; split the batch");
    DetArgs a;
    a.n = n; a.n_blocks = n_blocks; a.three = n_flavors == 3; a.dd = precision == COS_DET_DD;
    a.nsub = lattice == COS_LATTICE_HONEYCOMB ? 2 : 1; a.assign = 0; a.accumulate = 0;
    // kernel flavours 0, 1, 2; with two flavours the middle one is absent and caller flavour 1 takes slot 2
    const int flav[3] = {0, 1, n_flavors - 1};
    for (int f = 0; f < 3; ++f) {
        a.blk[f] = n_blocks == 1 ? 0 : flav[f];
        a.sigma[f] = shifts ? shifts[flav[f]] : 0.0;
    }
    uint32_t off = 0, b = 1;                          // level_off[k] = number of subsets larger than k
    a.level_off[n] = 0;
    for (int k = n; k >= 1; --k) {                    // b = binom(n, k)
        off += b;
        a.level_off[k - 1] = off;
        b = b * (uint32_t)k / (uint32_t)(n - k + 1);
    }
    a.G = G_dev; a.batch = batch; a.out = out_dev;
    // working-precision arrays first (16-byte elements need the alignment), the subset order behind them
    const size_t elem = a.dd ? 16 : 8, plane = ((size_t)1 << n) * (size_t)batch * elem;
    char* p = (char*)work_dev;
    a.minors = p; p += plane * n_blocks;
    a.H = p; p += plane;
    a.C = p; p += plane;
    a.order = (uint32_t*)p;
    cudaError_t e = launch_det_route(a, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "cos_det_eval: launch");
    return COS_OK;
}

// ---- cos_det_eval for callers that cannot allocate device memory (include/cos.h) ---------------------------------
// The scratch of the determinant route lives in this array instead of a caller's cudaMalloc'd buffer.  The name is
// usable as an address in DEVICE code only; on the host it is a stand-in object of the host program, so the launcher
// asks the runtime for the device address (cudaGetSymbolAddress), once per device, and hands that to the kernels.
static __device__ __align__(256) unsigned char g_det_static_scratch[COS_DET_STATIC_SCRATCH_BYTES];

namespace {
constexpr int kMaxStaticDevices = 64;
std::mutex g_det_static_mutex;
void* g_det_static_ptr[kMaxStaticDevices] = {};      // device address of g_det_static_scratch, per CUDA device

// Address of the array on the device that is current in this thread; looked up on the first call per device.
int det_static_scratch(void** ptr)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cos_det_eval_static: cudaGetDevice");
    if (dev < 0 || dev >= kMaxStaticDevices) return fail(COS_EUNSUPPORTED, "cos_det_eval_static: device ordinal above 63");
    std::lock_guard<std::mutex> lock(g_det_static_mutex);
    if (!g_det_static_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_det_static_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "cos_det_eval_static: cudaGetSymbolAddress");
        if (!p || ((size_t)p & 255u) != 0) return fail(COS_ECUDA, "cos_det_eval_static: bad address of the scratch array");
        g_det_static_ptr[dev] = p;
    }
    *ptr = g_det_static_ptr[dev];
    return COS_OK;
}
}  // namespace

int cos_det_eval_static(int n, int n_flavors, int n_blocks, int lattice, const double* shifts, int precision,
                        const double* G_dev, long long batch, double* out_dev, cos_stream stream)
{
    const long long need = cos_det_workspace_bytes(n, n_blocks, precision, batch);
    if (need > COS_DET_STATIC_SCRATCH_BYTES)
        return fail(COS_EUNSUPPORTED, "cos_det_eval_static: this problem needs " + std::to_string(need) +
                    " bytes of scratch, the built-in array holds " + std::to_string((long long)COS_DET_STATIC_SCRATCH_BYTES) +
                    "; split the batch or call cos_det_eval with a buffer of your own");
    // bad arguments (need < 0) and the empty batch never touch the scratch: cos_det_eval reports / returns before it
    // looks at the buffer
    if (need < 0 || batch == 0)
        return cos_det_eval(n, n_flavors, n_blocks, lattice, shifts, precision, G_dev, batch, out_dev, nullptr, 0, stream);
    void* scratch = nullptr;
    const int rc = det_static_scratch(&scratch);
    if (rc != COS_OK) return rc;
    // from here on: argument checks and kernel launches only (cos_det_eval allocates nothing)
    return cos_det_eval(n, n_flavors, n_blocks, lattice, shifts, precision, G_dev, batch, out_dev, scratch,
                        COS_DET_STATIC_SCRATCH_BYTES, stream);
}

int cos_equivalence_stats(int n, int n_flavors, int lattice, const double* shifts, int readout_envelope, int flags,
                          long long* out6)
{
    if (!out6) return fail(COS_EINVAL, "cos_equivalence_stats: out is NULL");
    if (n < 1 || n > COS_MAX_N || n_flavors < 1 || (lattice != COS_LATTICE_SQUARE && lattice != COS_LATTICE_HONEYCOMB) ||
        (readout_envelope != 0 && readout_envelope != n))
        return fail(COS_EINVAL, "cos_equivalence_stats: bad argument");
    const bool uniform_shift = (flags & COS_BUILD_UNIFORM_SHIFT) != 0;
    if (uniform_shift && !shifts) return fail(COS_EINVAL, "cos_equivalence_stats: COS_BUILD_UNIFORM_SHIFT needs shifts[0]");
    CompiledDag D;
    EquivalenceStats eq;
    std::string err = compile_dag(n, n_flavors, lattice == COS_LATTICE_HONEYCOMB ? 2 : 1, shifts, uniform_shift,
                                  readout_envelope == n, 0u, D, &eq);
    if (!err.empty()) return fail(is_unsupported(err) ? COS_EUNSUPPORTED : COS_ENOMEM, "cos_equivalence_stats: " + err);
    out6[0] = (long long)eq.n_states; out6[1] = (long long)eq.n_edges;
    out6[2] = (long long)eq.future_classes; out6[3] = (long long)eq.edges_after_future_merge;
    out6[4] = (long long)eq.past_classes; out6[5] = (long long)eq.edges_after_past_merge;
    return COS_OK;
}

int cos_debug_check_failures(long long* total, long long* by_kind)
{
    if (!total) return fail(COS_EINVAL, "cos_debug_check_failures: NULL argument");
    long long kinds[8];
    cudaError_t e = read_check_failures(total, kinds);
    if (e != cudaSuccess) return cuda_fail(e, "cos_debug_check_failures");
    if (by_kind) for (int k = 0; k < 8; ++k) by_kind[k] = kinds[k];
    return COS_OK;
}

int cos_measure_fp64_fma_peak(double* fma_per_s)
{
    if (!fma_per_s) return fail(COS_EINVAL, "cos_measure_fp64_fma_peak: NULL argument");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(COS_ECUDA, "no CUDA device");
    cudaError_t e = measure_fp64_fma(fma_per_s);
    if (e != cudaSuccess) return cuda_fail(e, "cos_measure_fp64_fma_peak");
    return COS_OK;
}

}  // extern "C"
