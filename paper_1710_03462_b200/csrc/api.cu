// api.cu -- the C ABI of include/soax.h: layout registry, container handles, argument checking, dispatch.
// Every step of the hot path runs in the kernels of the sibling .cu files; nothing here computes on the host.
#include <cstdlib>
#include <cstring>
#include <deque>
#include <mutex>
#include <new>
#include <string>

#include "common.cuh"
#include "expr.hpp"
#include "ops.hpp"

namespace soax {
std::atomic<int64_t> g_launches{0};
thread_local int g_last_cuda_error = 0;
Tuning g_tune;
}  // namespace soax

using namespace soax;

// ---- run-time descriptor of one compiled layout (generated from the typelist) -------------------------------
struct soax_layout {
    const char* name;
    int nfields, ncomp;
    const char* fname[kMaxComp];
    int fdtype[kMaxComp], fdim[kMaxComp], fbegin[kMaxComp];
    int cfield[kMaxComp], cdtype[kMaxComp], csize[kMaxComp];
    int (*step)(void* const*, int64_t, const soax_step_params*, cudaStream_t);
    int (*step_aos)(void*, int64_t, const soax_step_params*, int, cudaStream_t);
    int (*aos_to_soa)(void* const*, const void*, int64_t, cudaStream_t);
    int (*soa_to_aos)(void* const*, void*, int64_t, cudaStream_t);
    int (*gather_segments)(void* const*, const void*, const uint32_t*, const uint32_t*, int64_t, int64_t, cudaStream_t);
    int (*energy)(void* const*, int64_t, int, double, double, void*, double*, cudaStream_t);
    int (*bin_permute)(const BinArgs&, cudaStream_t);
    size_t (*bin_scratch)(int64_t, int, bool);
    int (*remove)(void* const*, void* const*, const uint8_t*, int64_t, int, void*, int64_t, int64_t*, int64_t*, cudaEvent_t, cudaStream_t);
    int (*gather_rows)(void* const*, int64_t, const uint32_t*, int64_t, void*, cudaStream_t);
    int (*remove_stable_noalloc)(void* const*, void* const*, const uint8_t*, int64_t, uint32_t, int64_t, int64_t*, cudaStream_t);
};

// A captured loop of `nlaunch` kernel launches, replayed while the call that made it is repeated unchanged: small
// (L2-resident) particle sets are launch-bound, and a graph replays its kernel nodes back to back without a host
// round trip per step.  Still one kernel launch and one full memory pass per step (Q14).  The key is the byte image of
// EVERYTHING the captured launches depend on (every component pointer, counts, parameters, tuning): a freed container
// whose address or slab is reused by a new one can therefore never replay the old graph.
struct GraphCache {
    cudaGraphExec_t exec = nullptr;
    std::string key;
    ~GraphCache() {}  // the exec is destroyed explicitly (soax_free / soax_expr_free); at thread exit the context may be gone
};

// True if `st` can be captured now: any stream but the legacy default stream that is not already being captured.
static bool capturable(cudaStream_t st) {
    if (st == nullptr || st == cudaStreamLegacy) return false;
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); return false; }
    return true;
}

// Replay the graph cached under `key`, capturing it first with nlaunch calls of enqueue(st) if the key changed.  Returns
// SOAX_OK with *done = true if the graph ran; *done = false if capture is not possible (the caller then issues the
// launches one by one).  `prepare` runs once before a capture (work that must not be captured, e.g. module loading).
template <class Prepare, class Enqueue>
static int replay_or_capture(GraphCache& g, const std::string& key, int32_t nlaunch, cudaStream_t st, Prepare&& prepare, Enqueue&& enqueue,
                             bool* done) {
    *done = false;
    if (!g.exec || g.key != key) {
        if (g.exec) { cudaGraphExecDestroy(g.exec); g.exec = nullptr; }
        SOAX_TRY(prepare());
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            int rc = SOAX_OK;
            for (int32_t i = 0; i < nlaunch && rc == SOAX_OK; ++i) rc = enqueue();
            const cudaError_t e = cudaStreamEndCapture(st, &graph);
            if (rc != SOAX_OK) { if (graph) cudaGraphDestroy(graph); cudaGetLastError(); return rc; }
            if (e == cudaSuccess && graph && cudaGraphInstantiate(&g.exec, graph, 0) != cudaSuccess) g.exec = nullptr;
            if (graph) cudaGraphDestroy(graph);
        }
        cudaGetLastError();
        if (g.exec) g.key = key;
    } else {
        g_launches.fetch_add(nlaunch, std::memory_order_relaxed);  // the replay launches the same nlaunch kernels
    }
    if (!g.exec) return SOAX_OK;
    SOAX_CUDA(cudaGraphLaunch(g.exec, st));
    *done = true;
    return SOAX_OK;
}

template <class T> static void key_add(std::string& k, const T& v) { k.append(reinterpret_cast<const char*>(&v), sizeof(T)); }

struct soax_container {
    const soax_layout* layout;
    int64_t n, capacity;
    void* comp[kMaxComp];
    uint64_t serial;  // unique per soax_alloc: part of every graph key
    GraphCache graph;
    // A live count that a kernel is still computing (soax_remove): the scan kernel stores it straight into `pin_n` (mapped
    // pinned host memory owned by the handle, -1 while nothing has landed) and the stream records `n_event`; the first later
    // call that needs the count on the host waits for that one event -- the count is ready after two small kernels, long
    // before the rows have moved.  One pending count per handle, resolved by one host thread: see soax.h.
    mutable bool n_pending = false;
    int64_t* pin_n = nullptr;
    cudaEvent_t n_event = nullptr;
};

// live particle count of a handle, resolving a pending one
static int64_t live(const soax_container* s) {
    if (s->n_pending) {
        const cudaError_t e = cudaEventSynchronize(s->n_event);
        const int64_t m = *s->pin_n;
        // The word holds -1 until the scan kernel has stored the count: a kernel that faulted, or an event that never really
        // fired, must not turn a stale word into the live count.  On failure the handle keeps the count it had and the CUDA
        // error is left for soax_last_cuda_error().
        if (e == cudaSuccess && m >= 0) const_cast<soax_container*>(s)->n = m > s->capacity ? s->capacity : m;  // STABLE into too small a destination holds the survivors that fit
        else if (e != cudaSuccess) cuda_fail(e);
        s->n_pending = false;
    }
    return s->n;
}
// A count that is still on its way targets pin_n: let it land (and be discarded) before the handle is given a new one, so that
// a later soax_remove on another stream never has two kernels writing that word unordered.
static void set_live(soax_container* s, int64_t n) {
    if (s->n_pending) cudaEventSynchronize(s->n_event);
    s->n = n;
    s->n_pending = false;
}

static std::string container_key(const soax_container* s) {
    std::string k;
    key_add(k, s->serial); key_add(k, s->layout); key_add(k, live(s)); key_add(k, s->capacity);
    k.append(reinterpret_cast<const char*>(s->comp), sizeof(void*) * s->layout->ncomp);
    key_add(k, g_tune);
    return k;
}

namespace {

template <class L>
soax_layout describe(const char* name) {
    soax_layout d{};
    d.name = name;
    d.nfields = L::nfields;
    d.ncomp = L::ncomp;
    for (int f = 0; f < L::nfields; ++f) {
        d.fname[f] = L::field_name(f);
        d.fdtype[f] = L::field_dtype(f);
        d.fdim[f] = L::field_dim(f);
        d.fbegin[f] = L::field_begin(f);
    }
    for (int c = 0; c < L::ncomp; ++c) {
        d.cfield[c] = L::comp_field(c);
        d.cdtype[c] = L::comp_dtype(c);
        d.csize[c] = L::comp_size(c);
    }
    d.step = &step_entry<L>;
    d.step_aos = &step_aos_entry<L>;
    d.aos_to_soa = &aos_to_soa_entry<L>;
    d.soa_to_aos = &soa_to_aos_entry<L>;
    d.gather_segments = &gather_segments_entry<L>;
    d.energy = &energy_entry<L>;
    d.bin_permute = &bin_permute_entry<L>;
    d.bin_scratch = &bin_scratch_bytes<L>;
    d.remove = &remove_entry<L>;
    d.gather_rows = &gather_rows_entry<L>;
    d.remove_stable_noalloc = &remove_stable_noalloc_entry<L>;
    return d;
}

const soax_layout* registry(int* count) {
#define X(L) describe<L>(#L),
    static const soax_layout table[] = {SOAX_FOR_EACH_LAYOUT(X)};
#undef X
    *count = (int)(sizeof(table) / sizeof(table[0]));
    return table;
}

size_t carve(const soax_layout* l, int64_t cap, void* slab, void** comps) {
    size_t off = 0;
    for (int c = 0; c < l->ncomp; ++c) {
        if (comps) comps[c] = static_cast<char*>(slab) + off;
        off += align_up((size_t)cap * (size_t)l->csize[c], kAlign);
    }
    return off > 0 ? off : kAlign;
}

inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

int ilog2_exact(int g) {
    for (int b = 0; b <= 6; ++b) if ((1 << b) == g) return b;
    return -1;
}

}  // namespace

extern "C" {

int soax_layout_define(const soax_field* fields, int32_t nfields, const soax_layout** out) {
    if (!fields || !out || nfields <= 0 || nfields > kMaxComp) return SOAX_ERR_INVALID_ARG;
    for (int f = 0; f < nfields; ++f)
        if (!fields[f].name || fields[f].dim <= 0 || dtype_size(fields[f].dtype) == 0) return SOAX_ERR_INVALID_ARG;
    int count = 0;
    const soax_layout* table = registry(&count);
    for (int i = 0; i < count; ++i) {
        const soax_layout& l = table[i];
        if (l.nfields != nfields) continue;
        bool same = true;
        for (int f = 0; f < nfields && same; ++f)
            same = std::strcmp(l.fname[f], fields[f].name) == 0 && l.fdtype[f] == fields[f].dtype && l.fdim[f] == fields[f].dim;
        if (same) { *out = &l; return SOAX_OK; }
    }
    return SOAX_ERR_UNKNOWN_LAYOUT;
}

// A run-time layout: the same descriptor as a compiled one, with no kernel families behind it (every family entry is
// null -> SOAX_ERR_UNSUPPORTED).  Descriptors live in a process-wide list and are never freed (handles are immutable
// and valid for the process lifetime, like the compiled ones); an identical field list returns the same handle.
namespace {
struct DynLayout {
    soax_layout desc{};
    std::string names[kMaxComp];
};
std::mutex g_dyn_mu;
std::deque<DynLayout> g_dyn;

bool is_identifier(const char* s) {
    if (!((*s >= 'a' && *s <= 'z') || (*s >= 'A' && *s <= 'Z') || *s == '_')) return false;
    for (; *s; ++s)
        if (!((*s >= 'a' && *s <= 'z') || (*s >= 'A' && *s <= 'Z') || (*s >= '0' && *s <= '9') || *s == '_')) return false;
    return true;
}
bool same_fields(const soax_layout& l, const soax_field* fields, int nfields) {
    if (l.nfields != nfields) return false;
    for (int f = 0; f < nfields; ++f)
        if (std::strcmp(l.fname[f], fields[f].name) != 0 || l.fdtype[f] != fields[f].dtype || l.fdim[f] != fields[f].dim) return false;
    return true;
}
}  // namespace

int soax_layout_define_dynamic(const soax_field* fields, int32_t nfields, const soax_layout** out) {
    const int rc = soax_layout_define(fields, nfields, out);  // a compiled instantiation wins: it has every kernel family
    if (rc != SOAX_ERR_UNKNOWN_LAYOUT) return rc;
    int ncomp = 0;
    for (int f = 0; f < nfields; ++f) {
        if (!is_identifier(fields[f].name)) return SOAX_ERR_INVALID_ARG;
        for (int g = 0; g < f; ++g)
            if (std::strcmp(fields[f].name, fields[g].name) == 0) return SOAX_ERR_INVALID_ARG;
        ncomp += fields[f].dim;
        if (ncomp > kMaxComp) return SOAX_ERR_INVALID_ARG;
    }
    std::lock_guard<std::mutex> lock(g_dyn_mu);
    for (const DynLayout& d : g_dyn)
        if (same_fields(d.desc, fields, nfields)) { *out = &d.desc; return SOAX_OK; }
    g_dyn.emplace_back();  // deque: earlier descriptors never move
    DynLayout& d = g_dyn.back();
    d.desc.name = "dynamic";
    d.desc.nfields = nfields;
    d.desc.ncomp = ncomp;
    int c = 0;
    for (int f = 0; f < nfields; ++f) {
        d.names[f] = fields[f].name;
        d.desc.fname[f] = d.names[f].c_str();
        d.desc.fdtype[f] = fields[f].dtype;
        d.desc.fdim[f] = fields[f].dim;
        d.desc.fbegin[f] = c;
        for (int k = 0; k < fields[f].dim; ++k, ++c) {
            d.desc.cfield[c] = f;
            d.desc.cdtype[c] = fields[f].dtype;
            d.desc.csize[c] = dtype_size(fields[f].dtype);
        }
    }
    *out = &d.desc;
    return SOAX_OK;
}

int soax_layout_nfields(const soax_layout* l) { return l ? l->nfields : SOAX_ERR_INVALID_ARG; }
int soax_layout_ncomp(const soax_layout* l) { return l ? l->ncomp : SOAX_ERR_INVALID_ARG; }

int soax_layout_comp(const soax_layout* l, int32_t c, int32_t* field, int32_t* comp_in_field, int32_t* dtype) {
    if (!l || c < 0 || c >= l->ncomp) return SOAX_ERR_INVALID_ARG;
    if (field) *field = l->cfield[c];
    if (comp_in_field) *comp_in_field = c - l->fbegin[l->cfield[c]];
    if (dtype) *dtype = l->cdtype[c];
    return SOAX_OK;
}

int soax_layout_aos(const soax_layout* l, int32_t packed, size_t* stride, size_t* comp_offsets) {
    if (!l) return SOAX_ERR_INVALID_ARG;
    size_t off = 0, maxal = 1;
    for (int c = 0; c < l->ncomp; ++c) {
        const size_t sz = (size_t)l->csize[c];
        if (!packed) { off = align_up(off, sz); if (sz > maxal) maxal = sz; }
        if (comp_offsets) comp_offsets[c] = off;
        off += sz;
    }
    if (!packed) off = align_up(off, maxal);
    if (stride) *stride = off;
    return SOAX_OK;
}

size_t soax_slab_bytes(const soax_layout* l, int64_t capacity) {
    if (!l || capacity < 0) return 0;
    return carve(l, capacity, nullptr, nullptr);
}

int soax_alloc(const soax_layout* l, int64_t n, int64_t capacity, void* dev_slab, size_t slab_bytes, soax_t** out) {
    if (!l || !out || n < 0 || capacity < n || !dev_slab || !aligned(dev_slab, kAlign)) return SOAX_ERR_INVALID_ARG;
    if (slab_bytes < carve(l, capacity, nullptr, nullptr)) return SOAX_ERR_ALLOC;
    soax_container* s = new (std::nothrow) soax_container();
    if (!s) return SOAX_ERR_ALLOC;
    s->layout = l;
    set_live(s, n);
    s->capacity = capacity;
    static std::atomic<uint64_t> next_serial{1};
    s->serial = next_serial.fetch_add(1, std::memory_order_relaxed);
    carve(l, capacity, dev_slab, s->comp);
    *out = s;
    return SOAX_OK;
}

int soax_free(soax_t* s) {
    if (!s) return SOAX_ERR_INVALID_ARG;
    if (s->graph.exec) cudaGraphExecDestroy(s->graph.exec);
    if (s->n_event) { cudaEventSynchronize(s->n_event); cudaEventDestroy(s->n_event); }  // a pending count copy targets pin_n
    if (s->pin_n) cudaFreeHost(s->pin_n);
    delete s;
    return SOAX_OK;
}

int64_t soax_size(const soax_t* s) { return s ? live(s) : (int64_t)SOAX_ERR_INVALID_ARG; }

int soax_resize(soax_t* s, int64_t n) {
    if (!s || n < 0 || n > s->capacity) return SOAX_ERR_INVALID_ARG;
    set_live(s, n);
    return SOAX_OK;
}

int soax_field_ptr(const soax_t* s, int32_t field, int32_t comp, void** dev_ptr) {
    if (!s || !dev_ptr || field < 0 || field >= s->layout->nfields) return SOAX_ERR_INVALID_ARG;
    if (comp < 0 || comp >= s->layout->fdim[field]) return SOAX_ERR_UNSUPPORTED;  // pos(42) on a 3-vector
    *dev_ptr = s->comp[s->layout->fbegin[field] + comp];
    return SOAX_OK;
}

int soax_upload(soax_t* s, const void* const* host_comps, int64_t n, void* stream) {
    if (!s || !host_comps || n < 0 || n > s->capacity) return SOAX_ERR_INVALID_ARG;
    for (int c = 0; c < s->layout->ncomp; ++c)
        if (host_comps[c] && n > 0)
            SOAX_CUDA(cudaMemcpyAsync(s->comp[c], host_comps[c], (size_t)n * s->layout->csize[c], cudaMemcpyHostToDevice,
                                      (cudaStream_t)stream));
    set_live(s, n);
    return SOAX_OK;
}

int soax_download(const soax_t* s, void* const* host_comps, int64_t n, void* stream) {
    if (!s || !host_comps || n < 0 || n > live(s)) return SOAX_ERR_INVALID_ARG;
    for (int c = 0; c < s->layout->ncomp; ++c)
        if (host_comps[c] && n > 0)
            SOAX_CUDA(cudaMemcpyAsync(host_comps[c], s->comp[c], (size_t)n * s->layout->csize[c], cudaMemcpyDeviceToHost,
                                      (cudaStream_t)stream));
    return SOAX_OK;
}

int soax_step(soax_t* s, const soax_step_params* p, int32_t nsteps, void* stream) {
    if (!s || !p || nsteps < 0) return SOAX_ERR_INVALID_ARG;
    if (!s->layout->step) return SOAX_ERR_UNSUPPORTED;  // run-time layout: no compiled kernel families
    cudaStream_t st = (cudaStream_t)stream;
    auto one = [&] { return s->layout->step(s->comp, live(s), p, st); };
    if (g_tune.step_graph && nsteps >= 2 && live(s) > 0 && capturable(st)) {
        std::string key = container_key(s);
        key_add(key, *p); key_add(key, nsteps);
        bool done = false;
        SOAX_TRY(replay_or_capture(s->graph, key, nsteps, st, [] { return SOAX_OK; }, one, &done));
        if (done) return SOAX_OK;
    }
    for (int32_t i = 0; i < nsteps; ++i) SOAX_TRY(one());
    return SOAX_OK;
}

int soax_step_aos(const soax_layout* l, void* dev_aos, int64_t n, const soax_step_params* p, int32_t nsteps,
                  int32_t variant, void* stream) {
    if (!l || !p || nsteps < 0 || n < 0 || (n > 0 && !dev_aos) || !aligned(dev_aos, 16)) return SOAX_ERR_INVALID_ARG;
    if (!l->step_aos) return SOAX_ERR_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    auto one = [&] { return l->step_aos(dev_aos, n, p, variant, st); };
    // Same graph replay as soax_step, so that the AoS baseline is timed under the same launch mechanism as the SoA
    // path.  There is no container to keep the graph with: one entry per host thread, keyed by the whole call.
    static thread_local GraphCache g;
    if (g_tune.step_graph && nsteps >= 2 && n > 0 && capturable(st)) {
        std::string key;
        key_add(key, l); key_add(key, dev_aos); key_add(key, n); key_add(key, *p); key_add(key, nsteps); key_add(key, variant); key_add(key, g_tune);
        bool done = false;
        SOAX_TRY(replay_or_capture(g, key, nsteps, st, [] { return SOAX_OK; }, one, &done));
        if (done) return SOAX_OK;
    }
    for (int32_t i = 0; i < nsteps; ++i) SOAX_TRY(one());
    return SOAX_OK;
}

int soax_aos_to_soa(soax_t* dst, const void* dev_aos, int64_t n, void* stream) {
    if (!dst || n < 0 || n > dst->capacity || (n > 0 && !dev_aos) || !aligned(dev_aos, 16)) return SOAX_ERR_INVALID_ARG;
    if (!dst->layout->aos_to_soa) return SOAX_ERR_UNSUPPORTED;
    set_live(dst, n);
    return n == 0 ? SOAX_OK : dst->layout->aos_to_soa(dst->comp, dev_aos, n, (cudaStream_t)stream);
}

int soax_soa_to_aos(const soax_t* src, void* dev_aos, int64_t n, void* stream) {
    if (!src || n < 0 || n > live(src) || (n > 0 && !dev_aos) || !aligned(dev_aos, 16)) return SOAX_ERR_INVALID_ARG;
    if (!src->layout->soa_to_aos) return SOAX_ERR_UNSUPPORTED;
    return n == 0 ? SOAX_OK : src->layout->soa_to_aos(const_cast<void* const*>(src->comp), dev_aos, n, (cudaStream_t)stream);
}

int soax_gather_segments_aos(soax_t* dst, const void* dev_aos, const uint32_t* dev_seg_dst, const uint32_t* dev_seg_src, int64_t nseg,
                             int64_t n, void* stream) {
    if (!dst || n < 0 || nseg < 0 || n > dst->capacity || n >= ((int64_t)1 << 32)) return SOAX_ERR_INVALID_ARG;
    if (n > 0 && (!dev_aos || !dev_seg_dst || !dev_seg_src || nseg == 0 || !aligned(dev_aos, 16) || !aligned(dev_seg_dst, 4) || !aligned(dev_seg_src, 4)))
        return SOAX_ERR_INVALID_ARG;
    if (!dst->layout->gather_segments) return SOAX_ERR_UNSUPPORTED;
    set_live(dst, n);
    return dst->layout->gather_segments(dst->comp, dev_aos, dev_seg_dst, dev_seg_src, nseg, n, (cudaStream_t)stream);
}

size_t soax_energy_scratch_bytes(void) { return kEnergyScratchBytes; }

int soax_reduce_energy(const soax_t* s, int32_t kind, double k, double center, void* dev_scratch, size_t scratch_bytes,
                       double* dev_out, void* stream) {
    if (!s || !dev_scratch || !dev_out || !aligned(dev_scratch, 8) || !aligned(dev_out, 8)) return SOAX_ERR_INVALID_ARG;
    if (scratch_bytes < kEnergyScratchBytes) return SOAX_ERR_ALLOC;
    if (!s->layout->energy) return SOAX_ERR_UNSUPPORTED;
    return s->layout->energy(const_cast<void* const*>(s->comp), live(s), kind, k, center, dev_scratch, dev_out,
                             (cudaStream_t)stream);
}

size_t soax_scratch_bytes(const soax_layout* l, int64_t n, int32_t grid_dim) {
    if (!l || n < 0 || ilog2_exact(grid_dim) < 0 || !l->bin_scratch) return 0;
    return l->bin_scratch(n, ilog2_exact(grid_dim), false);
}
size_t soax_scratch_bytes_inplace(const soax_layout* l, int64_t n, int32_t grid_dim) {
    if (!l || n < 0 || ilog2_exact(grid_dim) < 0 || !l->bin_scratch) return 0;
    return l->bin_scratch(n, ilog2_exact(grid_dim), true);
}

static int bin_permute_common(soax_t* src, soax_t* dst, bool inplace, int32_t grid_dim, double drift_dt, uint32_t* dev_counts,
                              uint32_t* dev_offsets, uint32_t* dev_perm, double* dev_kinetic, void* dev_scratch, size_t scratch_bytes,
                              void* stream) {
    if (!src || !dst || src == dst || src->layout != dst->layout || !dev_scratch || !aligned(dev_scratch, kAlign))
        return SOAX_ERR_INVALID_ARG;
    const int log2g = ilog2_exact(grid_dim);
    if (log2g < 0 || dst->capacity < live(src)) return SOAX_ERR_INVALID_ARG;
    if (!src->layout->bin_permute) return SOAX_ERR_UNSUPPORTED;
    for (int c = 0; c < src->layout->ncomp; ++c)
        if (src->comp[c] == dst->comp[c]) return SOAX_ERR_INVALID_ARG;
    if (live(src) >= ((int64_t)1 << 32)) return SOAX_ERR_UNSUPPORTED;
    const size_t need = src->layout->bin_scratch(live(src), log2g, inplace);
    if (need == 0) return SOAX_ERR_UNSUPPORTED;
    if (scratch_bytes < need) return SOAX_ERR_ALLOC;
    BinArgs a{src->comp, dst->comp, live(src), log2g, drift_dt, dev_counts, dev_offsets, dev_perm, dev_kinetic,
              dev_scratch, scratch_bytes, inplace};
    if (!inplace) set_live(dst, live(src));
    return src->layout->bin_permute(a, (cudaStream_t)stream);
}

int soax_bin_permute(soax_t* src, soax_t* dst, int32_t grid_dim, double drift_dt, uint32_t* dev_counts,
                     uint32_t* dev_offsets, uint32_t* dev_perm, double* dev_kinetic, void* dev_scratch,
                     size_t scratch_bytes, void* stream) {
    return bin_permute_common(src, dst, false, grid_dim, drift_dt, dev_counts, dev_offsets, dev_perm, dev_kinetic, dev_scratch,
                              scratch_bytes, stream);
}
int soax_bin_permute_inplace(soax_t* s, soax_t* work, int32_t grid_dim, double drift_dt, uint32_t* dev_counts,
                             uint32_t* dev_offsets, uint32_t* dev_perm, double* dev_kinetic, void* dev_scratch,
                             size_t scratch_bytes, void* stream) {
    return bin_permute_common(s, work, true, grid_dim, drift_dt, dev_counts, dev_offsets, dev_perm, dev_kinetic, dev_scratch,
                              scratch_bytes, stream);
}

// ---- NEXT-3: container operations (container_kernels.cu) ------------------------------------------------------------
size_t soax_remove_scratch_bytes(int64_t n) { return n < 0 ? 0 : remove_scratch_bytes(n); }

int soax_remove(soax_t* s, soax_t* dst, const uint8_t* dev_kill, int32_t mode, void* dev_scratch, size_t scratch_bytes,
                int64_t* host_new_n, void* stream) {
    if (!s) return SOAX_ERR_INVALID_ARG;
    const int64_t n = live(s);
    if ((n > 0 && (!dev_kill || !dev_scratch)) || !aligned(dev_scratch, kAlign)) return SOAX_ERR_INVALID_ARG;
    const int32_t base_mode = mode & ~SOAX_REMOVE_KEEP_FLAGGED;  // KEEP_FLAGGED: the mask marks the particles that stay
    if (base_mode != SOAX_REMOVE_SWAP_LAST && base_mode != SOAX_REMOVE_STABLE) return SOAX_ERR_INVALID_ARG;
    if (n >= ((int64_t)1 << 32) || !s->layout->remove) return SOAX_ERR_UNSUPPORTED;
    if (base_mode == SOAX_REMOVE_SWAP_LAST) {
        if (dst) return SOAX_ERR_INVALID_ARG;  // in place
    } else {
        if (!dst || dst == s || dst->layout != s->layout) return SOAX_ERR_INVALID_ARG;
        for (int c = 0; c < s->layout->ncomp; ++c)
            if (s->comp[c] == dst->comp[c]) return SOAX_ERR_INVALID_ARG;
    }
    if (n > 0 && scratch_bytes < remove_scratch_bytes(n)) return SOAX_ERR_ALLOC;
    soax_container* target = base_mode == SOAX_REMOVE_SWAP_LAST ? s : dst;
    if (n == 0) {
        if (host_new_n) *host_new_n = 0;
        set_live(target, 0);
        return SOAX_OK;
    }
    // The count travels through an event this call records and a later call waits for on the host: inside a stream capture
    // the event would never fire and the handle would read a stale word.
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing((cudaStream_t)stream, &cs) != cudaSuccess) { cudaGetLastError(); cs = cudaStreamCaptureStatusNone; }
    if (cs != cudaStreamCaptureStatusNone) return SOAX_ERR_UNSUPPORTED;
    if (!target->pin_n) {  // the event first: a handle never has the word without the event that guards it
        cudaEvent_t ev = nullptr;
        SOAX_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
        int64_t* word = nullptr;
        const cudaError_t e = cudaHostAlloc(reinterpret_cast<void**>(&word), sizeof(int64_t), cudaHostAllocMapped | cudaHostAllocPortable);
        if (e != cudaSuccess) { cudaEventDestroy(ev); return cuda_fail(e); }
        target->n_event = ev;
        target->pin_n = word;
    } else if (target->n_pending) {
        live(target);  // an earlier pending count still targets pin_n: let it land before the word is reused
    }
    *target->pin_n = -1;  // "nothing has landed yet" (the kernels of this call are enqueued after this store)
    SOAX_TRY(s->layout->remove(s->comp, dst ? dst->comp : nullptr, dev_kill, n, mode, dev_scratch, dst ? dst->capacity : 0,
                               target->pin_n, host_new_n, target->n_event, (cudaStream_t)stream));
    target->n_pending = true;
    return SOAX_OK;
}

// The one entry point that allocates nothing (see soax.h): no pinned word, no event, scratch inside the library image.  It reads
// the live count of s the usual way but leaves dst's count to the caller, who learns the survivor count from *dev_new_n.
int soax_remove_stable_noalloc(const soax_t* s, soax_t* dst, const uint8_t* dev_kill, int32_t keep_flagged, int64_t* dev_new_n,
                               void* stream) {
    if (!s || !dst || dst == s || dst->layout != s->layout || !dev_new_n || !aligned(dev_new_n, 8)) return SOAX_ERR_INVALID_ARG;
    const int64_t n = live(s);
    if (n > 0 && !dev_kill) return SOAX_ERR_INVALID_ARG;
    if (!s->layout->remove_stable_noalloc) return SOAX_ERR_UNSUPPORTED;
    for (int c = 0; c < s->layout->ncomp; ++c)
        if (s->comp[c] == dst->comp[c]) return SOAX_ERR_INVALID_ARG;
    if (n > SOAX_NOALLOC_MAX_N) return SOAX_ERR_TOO_LARGE;  // the work area compiled into the library holds counts for 2^24 rows
    if (n == 0) {
        SOAX_CUDA(cudaMemsetAsync(dev_new_n, 0, sizeof(int64_t), (cudaStream_t)stream));
        return SOAX_OK;
    }
    return s->layout->remove_stable_noalloc(s->comp, dst->comp, dev_kill, n, keep_flagged ? 1u : 0u, dst->capacity, dev_new_n,
                                            (cudaStream_t)stream);
}

int soax_push_back_aos(soax_t* s, const void* dev_aos, int64_t m, void* stream) {
    if (!s || m < 0 || (m > 0 && !dev_aos) || !aligned(dev_aos, 16)) return SOAX_ERR_INVALID_ARG;
    if (!s->layout->aos_to_soa) return SOAX_ERR_UNSUPPORTED;
    if (live(s) + m > s->capacity) return SOAX_ERR_ALLOC;  // the caller owns the memory: regrow = soax_alloc a larger slab + soax_copy
    if (m == 0) return SOAX_OK;
    void* tail[kMaxComp];
    for (int c = 0; c < s->layout->ncomp; ++c) tail[c] = static_cast<char*>(s->comp[c]) + (size_t)live(s) * s->layout->csize[c];
    SOAX_TRY(s->layout->aos_to_soa(tail, dev_aos, m, (cudaStream_t)stream));
    set_live(s, live(s) + m);
    return SOAX_OK;
}

int soax_get_elements(const soax_t* s, const uint32_t* dev_idx, int64_t m, void* dev_aos, void* stream) {
    if (!s || m < 0 || (m > 0 && (!dev_idx || !dev_aos)) || !aligned(dev_aos, 16) || !aligned(dev_idx, 4)) return SOAX_ERR_INVALID_ARG;
    if (!s->layout->gather_rows) return SOAX_ERR_UNSUPPORTED;
    return s->layout->gather_rows(const_cast<void* const*>(s->comp), live(s), dev_idx, m, dev_aos, (cudaStream_t)stream);
}

int soax_copy(soax_t* dst, const soax_t* src, void* stream) {
    if (!dst || !src || dst == src || dst->layout != src->layout) return SOAX_ERR_INVALID_ARG;
    if (dst->capacity < live(src)) return SOAX_ERR_ALLOC;
    for (int c = 0; c < src->layout->ncomp; ++c)
        if (live(src) > 0)
            SOAX_CUDA(cudaMemcpyAsync(dst->comp[c], src->comp[c], (size_t)live(src) * src->layout->csize[c], cudaMemcpyDeviceToDevice,
                                      (cudaStream_t)stream));
    set_live(dst, live(src));
    return SOAX_OK;
}

// ---- NEXT-2: fused element-wise programs (expr.cu) ----------------------------------------------------------------
struct soax_expr {
    CompiledExpr* impl;
    const soax_layout* layout;
    GraphCache graph;  // captured nsteps-launch loop, replayed while the call is the same (as soax_step does)
};

static int expr_compile_any(const soax_layout* l, const char* source, const char* const* scalar_names, int32_t nscalars, int kind,
                            soax_expr** out) {
    if (!l || !source || !out || nscalars < 0 || nscalars > 16 || (nscalars > 0 && !scalar_names)) return SOAX_ERR_INVALID_ARG;
    ExprLayoutInfo info{};
    info.nfields = l->nfields;
    info.ncomp = l->ncomp;
    for (int f = 0; f < l->nfields; ++f) { info.fname[f] = l->fname[f]; info.fdim[f] = l->fdim[f]; info.fbegin[f] = l->fbegin[f]; }
    for (int c = 0; c < l->ncomp; ++c) { info.cdtype[c] = l->cdtype[c]; info.csize[c] = l->csize[c]; }
    CompiledExpr* impl = nullptr;
    SOAX_TRY(expr_compile(info, l, source, scalar_names, nscalars, kind, &impl));
    soax_expr* e = new (std::nothrow) soax_expr();
    if (!e) { expr_free(impl); return SOAX_ERR_ALLOC; }
    e->impl = impl;
    e->layout = l;
    *out = e;
    return SOAX_OK;
}

int soax_expr_compile(const soax_layout* l, const char* source, const char* const* scalar_names, int32_t nscalars,
                      soax_expr** out) {
    return expr_compile_any(l, source, scalar_names, nscalars, 0, out);
}

int soax_expr_compile_sum(const soax_layout* l, const char* expression, const char* const* scalar_names, int32_t nscalars,
                          soax_expr** out) {
    return expr_compile_any(l, expression, scalar_names, nscalars, 1, out);
}

int soax_expr_compile_mask(const soax_layout* l, const char* condition, const char* const* scalar_names, int32_t nscalars,
                           soax_expr** out) {
    return expr_compile_any(l, condition, scalar_names, nscalars, 2, out);
}

int soax_expr_mask(const soax_t* s, soax_expr* e, const double* scalars, int32_t nscalars, uint8_t* dev_mask, void* stream) {
    if (!s || !e || nscalars < 0 || nscalars > 16 || (nscalars > 0 && !scalars)) return SOAX_ERR_INVALID_ARG;
    if (s->layout != e->layout) return SOAX_ERR_INVALID_ARG;
    const int64_t n = live(s);
    if (n > 0 && (!dev_mask || !aligned(dev_mask, 4))) return SOAX_ERR_INVALID_ARG;
    return expr_mask(e->impl, s->layout, const_cast<void* const*>(s->comp), n, scalars, nscalars, dev_mask, (cudaStream_t)stream);
}

int soax_expr_sum(const soax_t* s, soax_expr* e, const double* scalars, int32_t nscalars, void* dev_scratch, size_t scratch_bytes,
                  double* dev_out, void* stream) {
    if (!s || !e || !dev_scratch || !dev_out || !aligned(dev_scratch, 8) || !aligned(dev_out, 8) || nscalars < 0 || nscalars > 16)
        return SOAX_ERR_INVALID_ARG;
    if (s->layout != e->layout) return SOAX_ERR_INVALID_ARG;
    if (scratch_bytes < kEnergyScratchBytes) return SOAX_ERR_ALLOC;
    return expr_sum(e->impl, s->layout, const_cast<void* const*>(s->comp), live(s), scalars, nscalars, static_cast<double*>(dev_scratch),
                    dev_out, (cudaStream_t)stream);
}

int soax_expr_run(soax_t* s, soax_expr* e, const double* scalars, int32_t nscalars, int32_t nsteps, void* stream) {
    if (!s || !e || nsteps < 0 || nscalars < 0 || nscalars > 16 || (nscalars > 0 && !scalars)) return SOAX_ERR_INVALID_ARG;
    if (s->layout != e->layout) return SOAX_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    auto one = [&] { return expr_run(e->impl, s->layout, s->comp, live(s), scalars, nscalars, st); };
    if (g_tune.step_graph && nsteps >= 2 && live(s) > 0 && capturable(st)) {
        std::string key = container_key(s);  // every component pointer: a new container at a recycled address never matches
        key_add(key, nsteps); key_add(key, nscalars);
        if (nscalars) key.append(reinterpret_cast<const char*>(scalars), sizeof(double) * nscalars);
        bool done = false;
        // the first launch loads the generated code: do it (with n = 0) outside the capture
        SOAX_TRY(replay_or_capture(e->graph, key, nsteps, st,
                                   [&] { return expr_run(e->impl, s->layout, s->comp, 0, scalars, nscalars, st); }, one, &done));
        if (done) return SOAX_OK;
    }
    for (int32_t i = 0; i < nsteps; ++i) SOAX_TRY(one());
    return SOAX_OK;
}

int soax_expr_free(soax_expr* e) {
    if (!e) return SOAX_ERR_INVALID_ARG;
    if (e->graph.exec) cudaGraphExecDestroy(e->graph.exec);
    expr_free(e->impl);
    delete e;
    return SOAX_OK;
}

const char* soax_expr_error(void) { return expr_error(); }
const char* soax_expr_cuda_source(const soax_expr* e) { return e ? expr_cuda_source(e->impl) : nullptr; }
int soax_expr_traffic(const soax_expr* e, int32_t* bytes_read, int32_t* bytes_written) {
    if (!e) return SOAX_ERR_INVALID_ARG;
    int r = 0, w = 0;
    expr_traffic(e->impl, &r, &w);
    if (bytes_read) *bytes_read = r;
    if (bytes_written) *bytes_written = w;
    return SOAX_OK;
}

const char* soax_strerror(int status) {
    switch (status) {
        case SOAX_OK: return "ok";
        case SOAX_ERR_INVALID_ARG: return "invalid argument";
        case SOAX_ERR_UNKNOWN_LAYOUT: return "field list matches no compiled layout";
        case SOAX_ERR_UNSUPPORTED: return "operation not supported by this layout (missing field, wrong type or dimension)";
        case SOAX_ERR_ALLOC: return "buffer too small or host allocation failed";
        case SOAX_ERR_CUDA: return "CUDA runtime error (see soax_last_cuda_error)";
        case SOAX_ERR_TOO_LARGE: return "more particles than the built-in work area of soax_remove_stable_noalloc holds (SOAX_NOALLOC_MAX_N = 2^24): use soax_remove with your own scratch";
        default: return "unknown status";
    }
}

int soax_last_cuda_error(void) { return g_last_cuda_error; }
int64_t soax_launch_count(void) { return g_launches.load(); }
void soax_reset_launch_count(void) { g_launches.store(0); }

int soax_tune(const char* key, int64_t value) {
    if (!key) return SOAX_ERR_INVALID_ARG;
    const int v = (int)value;
    if (!std::strcmp(key, "step_ppt")) { if (v != 1 && v != 2 && v != 4) return SOAX_ERR_INVALID_ARG; g_tune.step_ppt = v; }
    else if (!std::strcmp(key, "step_block")) { if (v < 32 || v > 512 || v % 32) return SOAX_ERR_INVALID_ARG; g_tune.step_block = v; }
    else if (!std::strcmp(key, "step_persist")) { if (v < 0 || v > 64) return SOAX_ERR_INVALID_ARG; g_tune.step_persist = v; }
    else if (!std::strcmp(key, "aos_block")) { if (v < 32 || v > 1024 || v % 32) return SOAX_ERR_INVALID_ARG; g_tune.aos_block = v; }
    else if (!std::strcmp(key, "step_graph")) { if (v < 0 || v > 1) return SOAX_ERR_INVALID_ARG; g_tune.step_graph = v; }
    else if (!std::strcmp(key, "xpose_ring")) { if (v < 0 || v > 1) return SOAX_ERR_INVALID_ARG; g_tune.xpose_ring = v; }
    else if (!std::strcmp(key, "xpose_r")) { if (v != 0 && v != 1 && v != 2 && v != 4) return SOAX_ERR_INVALID_ARG; g_tune.xpose_r = v; }
    else if (!std::strcmp(key, "xpose_ns")) { if (v < 0 || v > 2) return SOAX_ERR_INVALID_ARG; g_tune.xpose_ns = v; }
    else if (!std::strcmp(key, "xpose_ctas")) { if (v < 0 || v > 8) return SOAX_ERR_INVALID_ARG; g_tune.xpose_ctas = v; }
    else if (!std::strcmp(key, "bin_bits")) { if (v < 0 || v > 9) return SOAX_ERR_INVALID_ARG; g_tune.bin_bits = v; }
    else if (!std::strcmp(key, "bin_cluster")) { if (v != 0 && v != 1 && v != 2 && v != 4 && v != 8 && v != 16) return SOAX_ERR_INVALID_ARG; g_tune.bin_cluster = v; }
    else if (!std::strcmp(key, "bin_pace_every")) { if (v < 0 || v > 8) return SOAX_ERR_INVALID_ARG; g_tune.bin_pace_every = v; }
    else if (!std::strcmp(key, "bin_pace")) { if (v < -1 || v > 16383) return SOAX_ERR_INVALID_ARG; g_tune.bin_pace = v; }
    else if (!std::strcmp(key, "bin_csync")) { if (v < 0 || v > 1) return SOAX_ERR_INVALID_ARG; g_tune.bin_csync = v; }
    else return SOAX_ERR_INVALID_ARG;
    return SOAX_OK;
}

}  // extern "C"
