// xs_api.cu -- the C ABI declared in include/xs.h.  Argument checking, workspace carving,
// host->device upload of the instance tables, and kernel launches; no arithmetic of the
// method lives here.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <new>

#include "xs_internal.h"

namespace {
thread_local std::string g_err;
int fail(int code, const std::string& msg)
{
    g_err = msg;
    return code;
}
int cuda_fail(int e, const char* where)
{
    g_err = std::string(where) + ": " + cudaGetErrorString((cudaError_t)e);
    return XS_ECUDA;
}
inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

int check_params(const xs_params* p)
{
    if (!p) return fail(XS_EINVAL, "params is null");
    if (p->n_spins < 3) return fail(XS_EINVAL, "n_spins must be >= 3");
    if (p->n_spins >= (1u << 28)) return fail(XS_EINVAL, "n_spins must be < 2^28");
    if (p->n_words == 0) return fail(XS_EINVAL, "n_words must be >= 1");
    if (p->n_instances == 0) return fail(XS_EINVAL, "n_instances must be >= 1");
    if (p->n_instances > 65535) return fail(XS_EINVAL, "n_instances must be <= 65535");
    if ((uint64_t)p->n_instances * p->n_words * 64 >= (1ull << 32))
        return fail(XS_EINVAL, "more than 2^32 clones in a batch");
    return XS_OK;
}
}  // namespace

namespace xs {
int xs_set_error(int code, const std::string& msg) { return fail(code, msg); }

DevLayout make_layout(const xs_params& p)
{
    DevLayout L;
    const size_t I = p.n_instances, N = p.n_spins, W = p.n_words;
    size_t o = 0;
    L.off_x = o;          o = align_up(o + I * N * W * 8, 256);
    L.off_first_hit = o;  o = align_up(o + I * W * 64 * 4, 256);
    L.off_adj = o;        o = align_up(o + I * N * sizeof(AdjRec), 256);
    L.off_clause = o;     o = align_up(o + I * N * sizeof(ClauseRec), 256);
    L.off_set_start = o;  o = align_up(o + I * (N + 1) * 4, 256);
    L.off_rec = o;        o = align_up(o + I * sizeof(xs_tts_rec), 256);
    L.off_seed = o;       o = align_up(o + I * 8, 256);
    L.off_det = o;        o = align_up(o + 2 * I * W * 8, 256);
    L.off_nsets = o;      o = align_up(o + I * 4, 256);
    L.off_crec = o;       o = align_up(o + I * (size_t)crec_entries(p) * sizeof(CRec), 256);
    L.off_cplace = o;     o = align_up(o + I * N * 4, 256);
    L.off_cbar = o;       o = align_up(o + I * 4, 256);
    L.off_cthr = o;       o = align_up(o + 8, 256);
    L.total = o;
    return L;
}
}  // namespace xs

using namespace xs;

// Launch geometry of a batch: the rule (choose_geometry), then the kernels with host-built tables
// (clause-word, latency).  Per-clone noise exists on the clause-word kernel (full lists) and on the
// streaming kernel only: a batch that the clause-word kernel does not take streams.
static int settle_geometry(xs_batch* b, void* stream)
{
    std::string err;
    b->p.flags = b->flags0;
    if (!choose_geometry(*b, b->geom, err)) return fail(XS_EINVAL, err);
    if (int e = clause_prepare(*b, stream)) return cuda_fail(e, "clause tables");
    if (int e = warp_prepare(*b, stream)) return cuda_fail(e, "latency kernel tables");
    if (b->ft.per_clone && b->geom.regime == 0 && b->geom.variant != 2) {
        b->p.flags |= XS_FLAG_STREAMING;
        if (!choose_geometry(*b, b->geom, err)) return fail(XS_EINVAL, err);
    }
    return XS_OK;
}

extern "C" {

const char* xs_last_error(void) { return g_err.c_str(); }

int xs_workspace_bytes(const xs_params* p, size_t* device_bytes)
{
    if (int rc = check_params(p)) return rc;
    if (!device_bytes) return fail(XS_EINVAL, "device_bytes is null");
    *device_bytes = make_layout(*p).total;
    return XS_OK;
}

static int finish_create(xs_batch* b, void* dev_ws, size_t ws_bytes, void* stream)
{
    const xs_params& p = b->p;
    const uint32_t I = p.n_instances, N = p.n_spins;
    b->lay = make_layout(p);
    if (ws_bytes < b->lay.total) return fail(XS_ENOMEM, "device workspace smaller than xs_workspace_bytes");
    if ((reinterpret_cast<uintptr_t>(dev_ws) & 255u) != 0) return fail(XS_EINVAL, "device workspace must be 256-byte aligned");
    char* ws = static_cast<char*>(dev_ws);
    b->ws = dev_ws;
    {
        // the device the workspace lives on (the caller's current device at create time)
        int dev = 0, sms = 0;
        if (cudaError_t e = cudaGetDevice(&dev)) return cuda_fail((int)e, "cudaGetDevice");
        if (cudaError_t e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev))
            return cuda_fail((int)e, "device attribute");
        b->device = dev;
        b->num_sms = sms > 0 ? (uint32_t)sms : 148u;
    }
    b->d.x = reinterpret_cast<uint64_t*>(ws + b->lay.off_x);
    b->d.first_hit = reinterpret_cast<uint32_t*>(ws + b->lay.off_first_hit);
    b->d.adj = reinterpret_cast<AdjRec*>(ws + b->lay.off_adj);
    b->d.clause = reinterpret_cast<ClauseRec*>(ws + b->lay.off_clause);
    b->d.set_start = reinterpret_cast<uint32_t*>(ws + b->lay.off_set_start);
    b->d.rec = reinterpret_cast<xs_tts_rec*>(ws + b->lay.off_rec);
    b->d.run_seed = reinterpret_cast<uint64_t*>(ws + b->lay.off_seed);
    b->d.det = reinterpret_cast<uint64_t*>(ws + b->lay.off_det);
    b->d.n_sets = reinterpret_cast<uint32_t*>(ws + b->lay.off_nsets);
    b->d.crec = reinterpret_cast<CRec*>(ws + b->lay.off_crec);
    b->d.cplace = reinterpret_cast<uint32_t*>(ws + b->lay.off_cplace);
    b->d.cbar = reinterpret_cast<uint32_t*>(ws + b->lay.off_cbar);
    b->d.cthr = reinterpret_cast<uint32_t*>(ws + b->lay.off_cthr);

    // host staging of the tables (pageable; the copies below are synchronous w.r.t. the host)
    std::vector<AdjRec> adj((size_t)I * N);
    std::vector<ClauseRec> cl((size_t)I * N);
    std::vector<uint32_t> ss((size_t)I * (N + 1), 0);
    std::vector<uint32_t> ns(I);
    std::vector<xs_tts_rec> rec(I);
    b->n_sets_max = 0;
    b->max_set_size = 0;
    for (uint32_t inst = 0; inst < I; ++inst) {
        const HostGraph& g = b->graphs[inst];
        const uint32_t n_sets = (uint32_t)g.set_start.size() - 1;
        ns[inst] = n_sets;
        b->n_sets_max = std::max(b->n_sets_max, n_sets);
        for (uint32_t s = 0; s <= n_sets; ++s) ss[(size_t)inst * (N + 1) + s] = g.set_start[s];
        for (uint32_t s = 0; s < n_sets; ++s)
            b->max_set_size = std::max(b->max_set_size, g.set_start[s + 1] - g.set_start[s]);
        for (uint32_t pos = 0; pos < N; ++pos) {
            const uint32_t v = g.order[pos];
            AdjRec& r = adj[(size_t)inst * N + pos];
            for (int q = 0; q < 6; ++q) r.nbr[q] = g.nbr[6ull * v + q];
            r.self = v;
            r.jbits = 0;
            for (int c = 0; c < 3; ++c) r.jbits |= (uint32_t)g.jbit[g.cls[3ull * v + c]] << c;
        }
        for (uint32_t t = 0; t < N; ++t)
            cl[(size_t)inst * N + t] = ClauseRec{g.tri[3ull * t], g.tri[3ull * t + 1], g.tri[3ull * t + 2], g.jbit[t]};
        rec[inst] = xs_tts_rec{0u, XS_NO_HIT, XS_NO_HIT, 0u, 0ull};
    }
    cudaStream_t st = (cudaStream_t)stream;
#define UP(dst, vec) \
    do { cudaError_t e_ = cudaMemcpyAsync(dst, (vec).data(), (vec).size() * sizeof((vec)[0]), cudaMemcpyHostToDevice, st); \
         if (e_ != cudaSuccess) return cuda_fail((int)e_, "upload"); } while (0)
    UP(b->d.adj, adj);
    UP(b->d.clause, cl);
    UP(b->d.set_start, ss);
    UP(b->d.n_sets, ns);
    UP(b->d.rec, rec);
    UP(b->d.run_seed, b->run_seeds);
#undef UP
    // staging vectors die at return: make sure the copies are done
    if (cudaError_t e = cudaStreamSynchronize(st)) return cuda_fail((int)e, "upload sync");

    // quasi-greedy table (0, w1, 1, 1) of L67 / L101 until xs_set_flip_table says otherwise
    b->ft = FlipTable{{0u, p.w1_threshold, 0u, 0u}, 0xCu, 0u, 0u, 0u};
    if (p.flags & XS_FLAG_CLONE_NOISE) {
        // per-clone noise: w1 = m / 128 with m the nearest integer
        b->ft.per_clone = 1u;
        b->ft.clone_m = (uint32_t)(((uint64_t)p.w1_threshold + (1ull << 24)) >> 25);
    }
    b->flags0 = b->p.flags;
    if (int rc = settle_geometry(b, stream)) return rc;
    if (int e = launch_init(*b, stream)) return cuda_fail(e, "init kernel");
    if (int e = launch_mark(*b, true, stream)) return cuda_fail(e, "mark kernel");
    if (int e = launch_finalize(*b, 0, stream)) return cuda_fail(e, "finalize kernel");
    return XS_OK;
}

int xs_create_instance(xs_batch** out, const xs_params* p, const uint64_t* graph_seeds,
                       const uint64_t* run_seeds, void* dev_ws, size_t ws_bytes, void* cuda_stream)
{
    if (int rc = check_params(p)) return rc;
    if (!out || !graph_seeds || !run_seeds || !dev_ws) return fail(XS_EINVAL, "null argument");
    xs_batch* b = new (std::nothrow) xs_batch();
    if (!b) return fail(XS_ENOMEM, "host allocation failed");
    b->p = *p;
    try {
        b->graphs.resize(p->n_instances);
        b->run_seeds.assign(run_seeds, run_seeds + p->n_instances);
        for (uint32_t i = 0; i < p->n_instances; ++i) {
            std::string err;
            if (!build_graph_from_seed(p->n_spins, graph_seeds[i], (p->flags & XS_FLAG_GAUGE) != 0,
                                       p->set_cap, (p->flags & XS_FLAG_BALANCED) != 0,
                                       b->graphs[i], err)) {
                delete b;
                return fail(XS_EINVAL, err);
            }
        }
        const int rc = finish_create(b, dev_ws, ws_bytes, cuda_stream);
        if (rc != XS_OK) { delete b; return rc; }
    } catch (const std::bad_alloc&) {
        delete b;
        return fail(XS_ENOMEM, "host allocation failed");
    }
    *out = b;
    return XS_OK;
}

int xs_create_instance_from_arrays(xs_batch** out, const xs_params* p, const uint32_t* tri,
                                   const uint8_t* jbit, const uint32_t* order,
                                   const uint32_t* set_size, const uint32_t* n_sets,
                                   uint32_t n_sets_max, const uint64_t* run_seeds, void* dev_ws,
                                   size_t ws_bytes, void* cuda_stream)
{
    if (int rc = check_params(p)) return rc;
    if (!out || !tri || !jbit || !order || !set_size || !n_sets || !run_seeds || !dev_ws)
        return fail(XS_EINVAL, "null argument");
    xs_batch* b = new (std::nothrow) xs_batch();
    if (!b) return fail(XS_ENOMEM, "host allocation failed");
    b->p = *p;
    try {
        const size_t N = p->n_spins;
        b->graphs.resize(p->n_instances);
        b->run_seeds.assign(run_seeds, run_seeds + p->n_instances);
        for (uint32_t i = 0; i < p->n_instances; ++i) {
            std::string err;
            if (n_sets[i] > n_sets_max ||
                !build_graph_from_arrays(p->n_spins, tri + 3 * N * i, jbit + N * i, order + N * i,
                                         set_size + (size_t)n_sets_max * i, n_sets[i], b->graphs[i], err)) {
                delete b;
                return fail(XS_EINVAL, err.empty() ? "n_sets exceeds n_sets_max" : err);
            }
        }
        const int rc = finish_create(b, dev_ws, ws_bytes, cuda_stream);
        if (rc != XS_OK) { delete b; return rc; }
    } catch (const std::bad_alloc&) {
        delete b;
        return fail(XS_ENOMEM, "host allocation failed");
    }
    *out = b;
    return XS_OK;
}

int xs_run_sweeps(xs_batch* b, uint64_t n_sweeps, void* cuda_stream)
{
    if (!b) return fail(XS_EINVAL, "batch is null");
    if (b->sweeps_issued + n_sweeps > 0xFFFFFFFEull)
        return fail(XS_ESTATE, "sweep counter would exceed 2^32 - 2");
    if (n_sweeps == 0) return XS_OK;
    if (int e = launch_sweeps(*b, (uint32_t)n_sweeps, cuda_stream)) return cuda_fail(e, "sweep kernel");
    if (int e = launch_finalize(*b, (uint32_t)n_sweeps, cuda_stream)) return cuda_fail(e, "finalize kernel");
    b->sweeps_issued += n_sweeps;
    return XS_OK;
}

int xs_set_flip_table(xs_batch* b, const uint64_t* thr4, void* cuda_stream)
{
    if (!b || !thr4) return fail(XS_EINVAL, "null argument");
    FlipTable ft{};
    for (int k = 0; k < 4; ++k) {
        if (thr4[k] > (1ull << 32)) return fail(XS_EINVAL, "threshold above 2^32");
        if (thr4[k] == (1ull << 32)) ft.always |= 1u << k;
        else ft.lo[k] = (uint32_t)thr4[k];
    }
    // the quasi-greedy form w = (0, w1 < 1, 1, 1) runs on the fast kernels
    ft.general = !(thr4[0] == 0 && ft.always == 0xCu);
    if (b->ft.per_clone) {
        if (thr4[0] != 0 || (ft.always & 0xCu) != 0xCu)
            return fail(XS_EINVAL, "per-clone noise supports the quasi-greedy form (0, w1, 1, 1) only");
        ft.general = 0u;
        ft.per_clone = 1u;
        ft.clone_m = (uint32_t)((thr4[1] + (1ull << 24)) >> 25);
    }
    b->ft = ft;
    if (!ft.general) b->p.w1_threshold = ft.lo[1];
    return settle_geometry(b, cuda_stream);
}

int xs_set_geometry(xs_batch* b, const xs_geometry* g, void* cuda_stream)
{
    if (!b) return fail(XS_EINVAL, "batch is null");
    xs_geometry rq{XS_GEOM_AUTO, 0, 0, 0, 0, 0};
    if (g) {
        rq = *g;
        if (rq.variant != XS_GEOM_AUTO && rq.variant > 3u) return fail(XS_EINVAL, "unknown kernel variant");
        if (rq.tile_words > 64u || (rq.tile_words & (rq.tile_words - 1u)))
            return fail(XS_EINVAL, "tile_words must be a power of two <= 64");
        if (rq.threads % 32u || rq.threads > 1024u) return fail(XS_EINVAL, "threads must be a multiple of 32, <= 1024");
        if (rq.words_per_lane > 2u) return fail(XS_EINVAL, "words_per_lane must be 0, 1 or 2");
    }
    const xs_geometry old = b->req;
    b->req = rq;
    if (int rc = settle_geometry(b, cuda_stream)) {
        b->req = old;
        settle_geometry(b, cuda_stream);
        return rc;
    }
    return XS_OK;
}

int xs_energy(xs_batch* b, int32_t* dev_out, void* cuda_stream)
{
    if (!b || !dev_out) return fail(XS_EINVAL, "null argument");
    if (int e = launch_energy(*b, dev_out, cuda_stream)) return cuda_fail(e, "energy kernel");
    return XS_OK;
}

int xs_tts(xs_batch* b, xs_tts_rec* host_out, void* cuda_stream)
{
    if (!b || !host_out) return fail(XS_EINVAL, "null argument");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (cudaError_t e = cudaMemcpyAsync(host_out, b->d.rec, sizeof(xs_tts_rec) * b->p.n_instances,
                                        cudaMemcpyDeviceToHost, st))
        return cuda_fail((int)e, "tts copy");
    if (cudaError_t e = cudaStreamSynchronize(st)) return cuda_fail((int)e, "tts sync");
    return XS_OK;
}

int xs_get_spins(xs_batch* b, uint64_t* dev_out, void* cuda_stream)
{
    if (!b || !dev_out) return fail(XS_EINVAL, "null argument");
    const size_t bytes = (size_t)b->p.n_instances * b->p.n_spins * b->p.n_words * 8;
    if (cudaError_t e = cudaMemcpyAsync(dev_out, b->d.x, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream))
        return cuda_fail((int)e, "get_spins");
    return XS_OK;
}

int xs_set_spins(xs_batch* b, const uint64_t* dev_in, void* cuda_stream)
{
    if (!b || !dev_in) return fail(XS_EINVAL, "null argument");
    const size_t bytes = (size_t)b->p.n_instances * b->p.n_spins * b->p.n_words * 8;
    if (cudaError_t e = cudaMemcpyAsync(b->d.x, dev_in, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream))
        return cuda_fail((int)e, "set_spins");
    if (int e = launch_mark(*b, true, cuda_stream)) return cuda_fail(e, "mark kernel");
    if (int e = launch_finalize(*b, 0, cuda_stream)) return cuda_fail(e, "finalize kernel");
    return XS_OK;
}

int xs_get_first_hit(xs_batch* b, uint32_t* dev_out, void* cuda_stream)
{
    if (!b || !dev_out) return fail(XS_EINVAL, "null argument");
    const size_t bytes = (size_t)b->p.n_instances * b->p.n_words * 64 * 4;
    if (cudaError_t e = cudaMemcpyAsync(dev_out, b->d.first_hit, bytes, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream))
        return cuda_fail((int)e, "get_first_hit");
    return XS_OK;
}

int xs_get_graph(const xs_batch* b, uint32_t inst, uint32_t* tri, uint8_t* jbit, uint32_t* order,
                 uint32_t* set_size, uint32_t* n_sets)
{
    if (!b) return fail(XS_EINVAL, "batch is null");
    if (inst >= b->p.n_instances) return fail(XS_EINVAL, "instance index out of range");
    const HostGraph& g = b->graphs[inst];
    const size_t N = b->p.n_spins;
    if (tri) std::memcpy(tri, g.tri.data(), 3 * N * sizeof(uint32_t));
    if (jbit) std::memcpy(jbit, g.jbit.data(), N);
    if (order) std::memcpy(order, g.order.data(), N * sizeof(uint32_t));
    const uint32_t ns = (uint32_t)g.set_start.size() - 1;
    if (set_size)
        for (uint32_t s = 0; s < ns; ++s) set_size[s] = g.set_start[s + 1] - g.set_start[s];
    if (n_sets) *n_sets = ns;
    return XS_OK;
}

int xs_clause_placement(uint32_t n_spins, uint64_t graph_seed, uint32_t flags, uint32_t set_cap,
                        uint32_t n_slots, uint32_t* task, uint32_t* place, uint32_t* n_rounds,
                        uint32_t* barrier_mask)
{
    if (n_spins < 3 || n_spins >= (1u << 24)) return fail(XS_EINVAL, "n_spins out of range");
    if (n_slots < 2 || n_slots > 256 || (n_slots & 1u)) return fail(XS_EINVAL, "n_slots must be even, 2..256");
    try {
        HostGraph g;
        std::string err;
        if (!build_graph_from_seed(n_spins, graph_seed, (flags & XS_FLAG_GAUGE) != 0, set_cap,
                                   (flags & XS_FLAG_BALANCED) != 0, g, err))
            return fail(XS_EINVAL, err);
        const uint32_t rounds = std::max(4u, clause_rounds(g, n_slots));
        std::vector<CRec> crec(2ull * n_spins, CRec{0u, 0u, 0u, 0xFFFFFFFFu});
        std::vector<uint32_t> cplace(n_spins);
        uint32_t bm = 0, mode = 0;
        if (!clause_placement(g, n_slots, rounds, crec.data(), cplace.data(), &bm, &mode))
            return fail(XS_EINVAL, "update order does not fit the clause-word kernel on this many slots, or no placement found");
        if (task) std::memcpy(task, crec.data(), (size_t)rounds * n_slots * sizeof(CRec));
        if (place) std::memcpy(place, cplace.data(), (size_t)n_spins * 4);
        if (n_rounds) *n_rounds = rounds;
        if (barrier_mask) *barrier_mask = bm;
    } catch (const std::bad_alloc&) {
        return fail(XS_ENOMEM, "host allocation failed");
    }
    return XS_OK;
}

int xs_generate_graph(uint32_t n_spins, uint64_t graph_seed, uint32_t flags, uint32_t set_cap,
                      uint32_t* tri, uint8_t* jbit, uint32_t* order, uint32_t* set_size,
                      uint32_t* n_sets, int32_t* attempt)
{
    if (n_spins < 3 || n_spins >= (1u << 28)) return fail(XS_EINVAL, "n_spins out of range");
    try {
        HostGraph g;
        std::string err;
        if (!build_graph_from_seed(n_spins, graph_seed, (flags & XS_FLAG_GAUGE) != 0, set_cap,
                                   (flags & XS_FLAG_BALANCED) != 0, g, err))
            return fail(XS_EINVAL, err);
        const size_t N = n_spins;
        if (tri) std::memcpy(tri, g.tri.data(), 3 * N * sizeof(uint32_t));
        if (jbit) std::memcpy(jbit, g.jbit.data(), N);
        if (order) std::memcpy(order, g.order.data(), N * sizeof(uint32_t));
        const uint32_t ns = (uint32_t)g.set_start.size() - 1;
        if (set_size)
            for (uint32_t s = 0; s < ns; ++s) set_size[s] = g.set_start[s + 1] - g.set_start[s];
        if (n_sets) *n_sets = ns;
        if (attempt) *attempt = g.attempt;
    } catch (const std::bad_alloc&) {
        return fail(XS_ENOMEM, "host allocation failed");
    }
    return XS_OK;
}

int xs_get_layout(const xs_batch* b, xs_layout* out)
{
    if (!b || !out) return fail(XS_EINVAL, "null argument");
    out->regime = b->geom.regime;
    out->tile_words = b->geom.T;
    out->threads = b->geom.threads;
    out->ctas = b->geom.ctas;
    out->smem_bytes = b->geom.smem;
    out->batch_sweeps = b->geom.batch;
    out->n_sets_max = b->n_sets_max;
    out->variant = b->geom.variant;
    return XS_OK;
}

int xs_destroy(xs_batch* b)
{
    delete b;
    return XS_OK;
}

}  // extern "C"
