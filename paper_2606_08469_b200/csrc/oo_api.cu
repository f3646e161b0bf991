// oo_api.cu — host side of liboo: the C ABI of include/oo.h.  Owns the device layouts (border-padded level-major
// atlases, dense + hop descent tables, the padded decoder image), validates what is uploaded, and dispatches kernels.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "oo_internal.h"

using namespace oo;

struct oo_ctx {
    int device = 0;
    int n_sms = 148;
    std::string err;
    std::string note;                      // informational: how the last upload / query resolved OO_PATH_AUTO (oo_last_note)
    cudaError_t sticky = cudaSuccess;      // a context-fatal CUDA error seen earlier (illegal address, launch failure, ...)
    oo_path path = OO_PATH_AUTO;
    FullModeH mode{0, 0, 0};
    oo_info info{};

    // tree
    bool have_tree = false;
    bool plan_ok = false;
    uint32_t tree_max_depth = 0;
    TreeParams T{};
    std::vector<void*> atlas_dev;          // library-owned padded atlases (unshifted base pointers)
    std::vector<uint64_t> level_slots;
    void* d_dense = nullptr;
    std::vector<void*> d_hop;
    void* d_child = nullptr;
    void* d_map_slot = nullptr;

    // mlp
    bool have_mlp = false;
    MlpParams M{};
    void* d_image = nullptr;
    void* d_image_tc = nullptr;

    // disparity predictor g_psi (f3)
    bool have_disp = false;
    GridParams G{};
    MlpParams MD{};
    void* d_grid = nullptr;
    void* d_disp_image = nullptr;

    // scene (f5)
    bool have_scene = false;
    void* d_spheres = nullptr;
    uint32_t n_spheres = 0;
    double scene_lo = 0.0, scene_hi = 1.0;

    // scratch
    uint64_t reserved = 0;
    void* d_feat = nullptr;    uint64_t feat_bytes = 0;   // feature rows of OO_PATH_GENERIC / OO_PATH_UNFUSED (sized by oo_reserve)
    uint32_t *d_keys_a = nullptr, *d_keys_b = nullptr, *d_idx_a = nullptr, *d_hist = nullptr;
    float *d_qx = nullptr, *d_qn = nullptr, *d_qw = nullptr, *d_qe = nullptr, *d_rgb = nullptr, *d_qd = nullptr;
    // OO_PRESORT_BIN: the binned copy of the queries and their original indices (allocated by oo_reserve, `reserved` rows)
    oo_presort presort = OO_PRESORT_AUTO;
    uint64_t bin_min = 1u << 18;           // batches below this proceed unsorted (the extra launches cost more than they save)
    // OO_PRESORT_AUTO: coherence samples of the recent calls (see kStatSlots).  The kernels write them to d_stat in device
    // memory; after a sampling call a copy to the pinned host array h_stat is enqueued on a library-owned side stream that
    // waits for the call's kernels, so the caller's stream carries nothing extra and the host never waits.
    unsigned long long* h_stat = nullptr;
    unsigned long long* d_stat = nullptr;
    cudaStream_t s_stat = nullptr;
    cudaEvent_t ev_stat = nullptr;
    bool armed = false;                    // the current call handed d_stat to a kernel
    uint32_t stat_seq = 0;                 // sequence number of the last sampling call
    bool auto_on = false;                  // current decision: bin the next large batch
    float coherence = 0.0f;                // mean distinct depth-4 cells per 32 consecutive queries, latest sample
    float *d_bx = nullptr, *d_bn = nullptr, *d_bw = nullptr, *d_be = nullptr;
    uint32_t *d_binv = nullptr, *d_bidx = nullptr, *d_btot = nullptr;   // d_btot: the bin pass's digit totals (zero between calls)
    float *d_brgb = nullptr, *d_bdisp = nullptr;

    // oo_query_host pipeline: copy-in and copy-out streams beside the caller's stream, one event pair per chunk
    static constexpr int kMaxChunks = 16;
    int host_chunks = 0;                   // oo_set_host_chunks: 0 = chosen from the batch size
    bool host_zero_copy = true;            // oo_query_host reads pinned host buffers in place when it can (oo_set_host_chunks(.., zero_copy))
    bool have_pipe = false;
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    cudaEvent_t ev_start = nullptr, ev_out = nullptr, ev_in[kMaxChunks] = {}, ev_k[kMaxChunks] = {};
};

namespace {

oo_status fail(oo_ctx* c, oo_status st, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf;
    return st;
}

// Errors after which the CUDA context is unusable: only these are latched (every later call on the oo_ctx then fails at
// once).  Anything else -- an allocation that did not fit, a launch configuration the device rejects, an invalid argument --
// is reported for the call that caused it, cleared, and the context stays usable.
bool is_fatal(cudaError_t e) {
    switch (e) {
        case cudaErrorIllegalAddress: case cudaErrorLaunchFailure: case cudaErrorIllegalInstruction: case cudaErrorMisalignedAddress:
        case cudaErrorInvalidAddressSpace: case cudaErrorInvalidPc: case cudaErrorHardwareStackError: case cudaErrorLaunchTimeout:
        case cudaErrorAssert: case cudaErrorECCUncorrectable: case cudaErrorDeviceUninitialized: case cudaErrorDevicesUnavailable:
            return true;
        default:
            return false;
    }
}

#define OO_CUDA(c, call)                                                                                      \
    do {                                                                                                      \
        cudaError_t e_ = (call);                                                                              \
        if (e_ != cudaSuccess) {                                                                              \
            (void)cudaGetLastError(); /* clear the thread's error state: the failure is reported here */      \
            if (is_fatal(e_)) (c)->sticky = e_;                                                               \
            return fail((c), e_ == cudaErrorMemoryAllocation ? OO_ERR_OOM : OO_ERR_CUDA, "%s: %s", #call,     \
                        cudaGetErrorString(e_));                                                              \
        }                                                                                                     \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) {
        cudaGetDevice(&prev);
        if (prev != dev) cudaSetDevice(dev);
        else prev = -1;
    }
    ~DeviceGuard() {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

void free_dev(void*& p) {
    if (p) cudaFree(p);
    p = nullptr;
}

void free_tree(oo_ctx* c) {
    for (void*& p : c->atlas_dev) free_dev(p);
    c->atlas_dev.clear();
    for (void*& p : c->d_hop) free_dev(p);
    c->d_hop.clear();
    free_dev(c->d_dense);
    free_dev(c->d_child);
    free_dev(c->d_map_slot);
    c->have_tree = false;
    c->plan_ok = false;
    c->info.node_table_bytes = c->info.atlas_bytes = 0;
}

void free_scratch(oo_ctx* c) {
    free_dev(c->d_feat);
    c->feat_bytes = 0;
    void** ps[] = {(void**)&c->d_keys_a, (void**)&c->d_keys_b, (void**)&c->d_idx_a, (void**)&c->d_hist, (void**)&c->d_qx,
                   (void**)&c->d_qn,     (void**)&c->d_qw,     (void**)&c->d_qe,    (void**)&c->d_rgb, (void**)&c->d_qd};
    for (void** p : ps) free_dev(*p);
    void** bs[] = {(void**)&c->d_bx, (void**)&c->d_bn, (void**)&c->d_bw, (void**)&c->d_be, (void**)&c->d_binv, (void**)&c->d_bidx, (void**)&c->d_brgb, (void**)&c->d_bdisp, (void**)&c->d_btot};
    for (void** p : bs) free_dev(*p);
    c->reserved = 0;
}

void free_pipe(oo_ctx* c) {
    if (c->s_h2d) cudaStreamDestroy(c->s_h2d);
    if (c->s_d2h) cudaStreamDestroy(c->s_d2h);
    if (c->ev_start) cudaEventDestroy(c->ev_start);
    if (c->ev_out) cudaEventDestroy(c->ev_out);
    for (int i = 0; i < oo_ctx::kMaxChunks; ++i) {
        if (c->ev_in[i]) cudaEventDestroy(c->ev_in[i]);
        if (c->ev_k[i]) cudaEventDestroy(c->ev_k[i]);
        c->ev_in[i] = c->ev_k[i] = nullptr;
    }
    c->s_h2d = c->s_d2h = nullptr;
    c->ev_start = c->ev_out = nullptr;
    c->have_pipe = false;
}

bool is_pow2(uint32_t v) { return v && !(v & (v - 1)); }

// Before the library launches anything: fail at once on a context that already saw a fatal error; a fatal error pending on
// the calling thread (whoever caused it, the CUDA context is gone) is latched and reported; a pending NON-fatal error of the
// thread -- some other library's rejected launch, say -- is not ours to report: it is cleared so that the check after our own
// launches sees only them.
oo_status check_before(oo_ctx* c) {
    if (c->sticky != cudaSuccess) return fail(c, OO_ERR_CUDA, "earlier CUDA failure: %s", cudaGetErrorString(c->sticky));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess && is_fatal(e)) {
        c->sticky = e;
        return fail(c, OO_ERR_CUDA, "asynchronous CUDA failure: %s", cudaGetErrorString(e));
    }
    return OO_OK;
}
// After the library's own launches: cudaGetLastError (which clears) reports what they produced.
oo_status check_after(oo_ctx* c) {
    const cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) return OO_OK;
    if (is_fatal(e)) c->sticky = e;
    return fail(c, OO_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(e));
}
// A launcher's return value: > 0 launches (counted), -1 no such kernel, kLaunchCudaError a CUDA call failed on the way.
oo_status launch_failed(oo_ctx* c, int n, const char* what) {
    if (n == kLaunchCudaError) {
        const cudaError_t e = cudaGetLastError();
        if (is_fatal(e)) c->sticky = e;
        return fail(c, OO_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
    }
    return fail(c, OO_ERR_UNSUPPORTED, "%s: no kernel for this shape", what);
}

oo_status check_queries(oo_ctx* c, const oo_queries* q, bool need_nrm) {
    if (!q) return fail(c, OO_ERR_INVALID_ARG, "queries is NULL");
    if (q->n == 0) return OO_OK;
    if (!q->x || !q->wo) return fail(c, OO_ERR_INVALID_ARG, "queries.x / queries.wo is NULL");
    if (need_nrm && !q->nrm) return fail(c, OO_ERR_INVALID_ARG, "queries.nrm is NULL");
    if (q->n_extra > OO_MAX_EXTRA) return fail(c, OO_ERR_INVALID_ARG, "n_extra %u > %d", q->n_extra, OO_MAX_EXTRA);
    if (need_nrm && q->n_extra && !q->extra) return fail(c, OO_ERR_INVALID_ARG, "n_extra > 0 but queries.extra is NULL");
    if (q->n >= (1ull << 32)) return fail(c, OO_ERR_UNSUPPORTED, "more than 2^32-1 queries per call");
    return OO_OK;
}

QueryParams make_qp(const oo_queries* q) {
    QueryParams Q{};
    Q.n = q->n; Q.x = q->x; Q.nrm = q->nrm; Q.wo = q->wo; Q.extra = q->extra; Q.n_extra = q->n_extra; Q.perm = q->perm;
    Q.disparity = q->disparity;
    return Q;
}

void count(oo_ctx* c, int launches) {
    if (launches > 0) {
        c->info.launches += (uint64_t)launches;
        c->info.query_launches += (uint64_t)launches;
    }
}

}  // namespace

// =====================================================================================================================

extern "C" OO_API oo_status oo_create(oo_ctx** out, int cuda_device) {
    if (!out) return OO_ERR_INVALID_ARG;
    *out = nullptr;
    oo_ctx* c = new (std::nothrow) oo_ctx();
    if (!c) return OO_ERR_OOM;
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || cuda_device < 0 || cuda_device >= n) {
        delete c;
        return OO_ERR_CUDA;
    }
    cudaDeviceProp prop{};
    e = cudaGetDeviceProperties(&prop, cuda_device);
    if (e != cudaSuccess || prop.major != 10) {   // kernels are sm_100a only
        delete c;
        return OO_ERR_CUDA;
    }
    c->device = cuda_device;
    c->n_sms = prop.multiProcessorCount;
    c->info.n_sms = (uint32_t)c->n_sms;
    {   // OO_PRESORT_AUTO: sample array on the device, its pinned host copy, the side stream and event that bring it over
        DeviceGuard g(cuda_device);
        const size_t bytes = kStatSlots * sizeof(unsigned long long);
        if (cudaMalloc((void**)&c->d_stat, bytes) == cudaSuccess && cudaMemset(c->d_stat, 0, bytes) == cudaSuccess &&
            cudaHostAlloc((void**)&c->h_stat, bytes, cudaHostAllocDefault) == cudaSuccess &&
            cudaStreamCreateWithFlags(&c->s_stat, cudaStreamNonBlocking) == cudaSuccess &&
            cudaEventCreateWithFlags(&c->ev_stat, cudaEventDisableTiming) == cudaSuccess) {
            memset(c->h_stat, 0, bytes);
        } else {
            (void)cudaGetLastError();
            c->presort = OO_PRESORT_NONE;      // AUTO has nothing to decide from
        }
    }
    *out = c;
    return OO_OK;
}

extern "C" OO_API void oo_destroy(oo_ctx* c) {
    if (!c) return;
    {
        DeviceGuard g(c->device);
        free_tree(c);
        free_dev(c->d_image);
        free_dev(c->d_image_tc);
        free_dev(c->d_spheres);
        free_dev(c->d_grid);
        free_dev(c->d_disp_image);
        free_scratch(c);
        free_pipe(c);
        if (c->s_stat) {
            cudaStreamSynchronize(c->s_stat);  // a copy into h_stat may still be in flight
            cudaStreamDestroy(c->s_stat);
        }
        if (c->ev_stat) cudaEventDestroy(c->ev_stat);
        if (c->h_stat) cudaFreeHost(c->h_stat);
        if (c->d_stat) cudaFree(c->d_stat);
    }
    delete c;
}

extern "C" OO_API const char* oo_last_error(const oo_ctx* c) { return c ? c->err.c_str() : "context is NULL"; }
extern "C" OO_API const char* oo_last_note(const oo_ctx* c) { return c ? c->note.c_str() : ""; }

extern "C" OO_API oo_status oo_set_path(oo_ctx* c, oo_path path) {
    if (!c) return OO_ERR_INVALID_ARG;
    if ((int)path < 0 || (int)path > (int)OO_PATH_FUSED_TC_TMEM) return fail(c, OO_ERR_INVALID_ARG, "unknown path %d", (int)path);
    c->path = path;
    return OO_OK;
}
extern "C" OO_API oo_status oo_set_presort(oo_ctx* c, oo_presort presort, uint64_t min_queries) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (presort != OO_PRESORT_NONE && presort != OO_PRESORT_BIN && presort != OO_PRESORT_AUTO) return fail(c, OO_ERR_INVALID_ARG, "unknown presort %d", (int)presort);
    if (presort == OO_PRESORT_AUTO && !c->ev_stat) return fail(c, OO_ERR_UNSUPPORTED, "OO_PRESORT_AUTO: the sample buffers could not be created on this context");
    c->presort = presort;
    c->bin_min = min_queries ? min_queries : (1u << 18);
    return OO_OK;
}

extern "C" OO_API oo_status oo_set_mode(oo_ctx* c, const oo_mode* m) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!m) return fail(c, OO_ERR_INVALID_ARG, "mode is NULL");
    if ((int)m->spatial < 0 || (int)m->spatial > (int)OO_SPATIAL_TRILINEAR8 || (int)m->lookup < 0 || (int)m->lookup > (int)OO_LOOKUP_SHIFTED ||
        (int)m->attrs < 0 || (int)m->attrs > (int)OO_ATTRS_PAPER)
        return fail(c, OO_ERR_INVALID_ARG, "unknown mode value (spatial %d, lookup %d, attrs %d)", (int)m->spatial, (int)m->lookup, (int)m->attrs);
    c->mode.tri8 = m->spatial == OO_SPATIAL_TRILINEAR8;
    c->mode.lookup = (uint32_t)m->lookup;
    c->mode.attrs_paper = m->attrs == OO_ATTRS_PAPER;
    return OO_OK;
}

extern "C" OO_API oo_status oo_get_info(const oo_ctx* c, oo_info* out) {
    if (!c || !out) return OO_ERR_INVALID_ARG;
    *out = c->info;
    out->hop_plan_ok = c->plan_ok ? 1u : 0u;
    out->full_query = c->mode.tri8 || c->mode.lookup || c->mode.attrs_paper || (c->have_tree && c->T.vertex) || (c->have_mlp && c->M.width != 64);
    out->n_neighbours = c->mode.tri8 ? 8u : 1u;
    out->presort_auto_on = c->auto_on ? 1u : 0u;
    out->coherence_x100 = (uint32_t)(c->coherence * 100.0f + 0.5f);
    return OO_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// oo_upload_tree
// ---------------------------------------------------------------------------------------------------------------------
extern "C" OO_API oo_status oo_upload_tree(oo_ctx* c, const oo_tree_desc* t, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!t) return fail(c, OO_ERR_INVALID_ARG, "tree is NULL");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g(c->device);
    // ---- validate the description
    if (t->n_nodes == 0 || !t->child || !t->depth || !t->map_slot) return fail(c, OO_ERR_INVALID_ARG, "empty tree or NULL node arrays");
    if (t->max_depth == 0 || t->max_depth > OO_MAX_DEPTH) return fail(c, OO_ERR_INVALID_ARG, "max_depth %u outside 1..%d", t->max_depth, OO_MAX_DEPTH);
    if (t->n_levels == 0 || t->n_levels > OO_MAX_LEVELS) return fail(c, OO_ERR_INVALID_ARG, "n_levels %u outside 1..%d", t->n_levels, OO_MAX_LEVELS);
    if (!t->level_depth || !t->level_res || !t->level_slots || !t->atlas) return fail(c, OO_ERR_INVALID_ARG, "NULL level arrays");
    if (t->dtype != OO_F16 && t->dtype != OO_F32) return fail(c, OO_ERR_INVALID_ARG, "unknown dtype");
    if (t->dirmap != OO_DIRMAP_TEXEL && t->dirmap != OO_DIRMAP_VERTEX) return fail(c, OO_ERR_INVALID_ARG, "unknown dirmap");
    const bool vertex = t->dirmap == OO_DIRMAP_VERTEX;
    const uint32_t esize = t->dtype == OO_F32 ? 4 : 2;
    const uint32_t texel_bytes = t->n_features * esize;
    if (texel_bytes != 16 && texel_bytes != 32 && texel_bytes != 64)
        return fail(c, OO_ERR_INVALID_ARG, "F*sizeof(dtype) = %u bytes; must be 16, 32 or 64", texel_bytes);
    const uint32_t L = t->n_levels;
    for (uint32_t l = 0; l < L; ++l) {
        if (t->level_depth[l] < 1 || t->level_depth[l] > t->max_depth) return fail(c, OO_ERR_INVALID_ARG, "level_depth[%u] = %u outside 1..max_depth", l, t->level_depth[l]);
        if (l && t->level_depth[l] <= t->level_depth[l - 1]) return fail(c, OO_ERR_INVALID_ARG, "level_depth must be strictly increasing");
        if (!is_pow2(t->level_res[l]) || t->level_res[l] < 2 || t->level_res[l] > 256) return fail(c, OO_ERR_INVALID_ARG, "level_res[%u] = %u: need a power of two in 2..256", l, t->level_res[l]);
        if (t->level_slots[l] && !t->atlas[l]) return fail(c, OO_ERR_INVALID_ARG, "atlas[%u] is NULL", l);
        if (((uintptr_t)t->atlas[l]) & 15) return fail(c, OO_ERR_INVALID_ARG, "atlas[%u] is not 16-byte aligned", l);
    }
    // ---- validate the nodes; per-depth local indices (used depth: map_slot; otherwise running count)
    const uint32_t N = t->n_nodes, D = t->max_depth;
    int level_of_depth[OO_MAX_DEPTH + 1];
    for (uint32_t d = 0; d <= D; ++d) level_of_depth[d] = -1;
    for (uint32_t l = 0; l < L; ++l) level_of_depth[t->level_depth[l]] = (int)l;
    if (t->depth[0] != 0) return fail(c, OO_ERR_INVALID_ARG, "node 0 must be the root (depth 0)");
    std::vector<int32_t> local(N);
    std::vector<uint32_t> depth_count(D + 1, 0);
    std::vector<std::vector<uint8_t>> seen(L);
    for (uint32_t l = 0; l < L; ++l) seen[l].assign(t->level_slots[l], 0);
    std::vector<uint8_t> has_parent(N, 0);
    for (uint32_t i = 0; i < N; ++i) {
        const uint32_t d = t->depth[i];
        if (d > D) return fail(c, OO_ERR_INVALID_ARG, "node %u: depth %u > max_depth", i, d);
        if (i && d == 0) return fail(c, OO_ERR_INVALID_ARG, "node %u: a second root", i);
        const int l = level_of_depth[d];
        if (l >= 0) {
            const int32_t s = t->map_slot[i];
            if (s < 0 || (uint32_t)s >= t->level_slots[l]) return fail(c, OO_ERR_INVALID_ARG, "node %u: map_slot %d outside level %d (%u slots)", i, s, l, t->level_slots[l]);
            if (seen[l][s]) return fail(c, OO_ERR_INVALID_ARG, "node %u: map_slot %d used twice in level %d", i, s, l);
            seen[l][s] = 1;
            local[i] = s;
        } else {
            if (t->map_slot[i] != -1) return fail(c, OO_ERR_INVALID_ARG, "node %u: map_slot must be -1 at an unused depth", i);
            local[i] = (int32_t)depth_count[d];
        }
        depth_count[d]++;
        for (int o = 0; o < 8; ++o) {
            const int32_t ch = t->child[(size_t)i * 8 + o];
            if (ch == -1) continue;
            if (ch <= 0 || (uint32_t)ch >= N) return fail(c, OO_ERR_INVALID_ARG, "node %u: child %d out of range", i, ch);
            if (t->depth[ch] != d + 1) return fail(c, OO_ERR_INVALID_ARG, "node %u (depth %u): child %d has depth %u", i, d, ch, (uint32_t)t->depth[ch]);
            if (has_parent[ch]) return fail(c, OO_ERR_INVALID_ARG, "node %d has two parents", ch);
            has_parent[ch] = 1;
        }
    }
    for (uint32_t i = 1; i < N; ++i)
        if (!has_parent[i]) return fail(c, OO_ERR_INVALID_ARG, "node %u is unreachable", i);

    // ---- replace the previous tree
    free_tree(c);
    TreeParams T{};
    T.n_levels = L; T.F = t->n_features; T.f32 = t->dtype == OO_F32; T.texel_bytes = texel_bytes;
    T.vertex = vertex ? 1u : 0u;
    T.depth_eff = t->level_depth[L - 1];
    T.scale_eff = (float)(1u << T.depth_eff);
    c->tree_max_depth = D;
    c->level_slots.assign(t->level_slots, t->level_slots + L);

    // ---- atlases: padded copies
    c->atlas_dev.assign(L, nullptr);
    uint64_t atlas_bytes = 0;
    int launches = 0;
    // vertex maps: number of boundary vertices the tying rewrote.  Freed on EVERY way out of this function (the early returns
    // below included: a failed upload on a usable context must not leave device memory behind).
    struct FreeAtExit { void* p = nullptr; ~FreeAtExit() { if (p) cudaFree(p); } } changed_owner;
    unsigned long long* d_changed = nullptr;
    if (vertex) {
        OO_CUDA(c, cudaMalloc(&changed_owner.p, sizeof(unsigned long long)));
        d_changed = (unsigned long long*)changed_owner.p;
        OO_CUDA(c, cudaMemsetAsync(d_changed, 0, sizeof(unsigned long long), stream));
    }
    for (uint32_t l = 0; l < L; ++l) {
        // texel maps: (R+2)^2 with the wrapped border; vertex maps: the (R+1)^2 vertices as given
        const uint32_t R = t->level_res[l], Rp = vertex ? R + 1 : R + 2;
        const uint64_t slots = std::max<uint64_t>(t->level_slots[l], 1);      // at least one (zero) map, so that the branch-free gather has an address
        const uint64_t map_bytes = (uint64_t)Rp * Rp * texel_bytes;
        const uint64_t lead = map_bytes;                                      // the all-zero map "slot -1" in front of slot 0
        const uint64_t bytes = lead + slots * map_bytes;
        if (bytes / 16 >= (1ull << 32)) return fail(c, OO_ERR_UNSUPPORTED, "level %u: %llu bytes of maps; a level is addressed in 32-bit units of 16 bytes (64 GB)", l, (unsigned long long)bytes);
        OO_CUDA(c, cudaMalloc(&c->atlas_dev[l], bytes));
        atlas_bytes += bytes;
        uint8_t* slot0 = (uint8_t*)c->atlas_dev[l] + lead;
        if (lead) OO_CUDA(c, cudaMemsetAsync(c->atlas_dev[l], 0, lead, stream));
        if (t->level_slots[l] == 0) OO_CUDA(c, cudaMemsetAsync(slot0, 0, slots * map_bytes, stream));
        else if (vertex) {
            OO_CUDA(c, cudaMemcpyAsync(slot0, t->atlas[l], slots * map_bytes, cudaMemcpyDeviceToDevice, stream));
            launches += launch_tie_vertex_borders(slot0, t->level_slots[l], R, texel_bytes, d_changed, stream);      // f2: P:125
        } else launches += launch_pad_atlas(t->atlas[l], slot0, t->level_slots[l], R, texel_bytes, stream);
        LevelParams& lv = T.lv[l];
        lv.atlas = slot0 + (vertex ? 0 : (uint64_t)(Rp + 1) * texel_bytes);
        lv.atlas_z = vertex ? nullptr : (const uint8_t*)c->atlas_dev[l];
        lv.map16 = (uint32_t)(map_bytes / 16);
        lv.tap16 = (Rp + 1) * texel_bytes / 16;
        lv.rp_f = (float)Rp;
        lv.half_r = 0.5f * (float)R;
        lv.off = 0.5f * (float)R - 0.5f;
        lv.R = R; lv.Rp = Rp;
        lv.map_bytes = Rp * Rp * texel_bytes;
        lv.row_bytes = Rp * texel_bytes;
        lv.depth = t->level_depth[l];
        lv.shift = T.depth_eff - lv.depth;
    }
    c->info.atlas_bytes = atlas_bytes;

    // ---- plain tables for the generic kernels
    uint64_t table_bytes = 0;
    OO_CUDA(c, cudaMalloc(&c->d_child, (size_t)N * 8 * 4));
    OO_CUDA(c, cudaMalloc(&c->d_map_slot, (size_t)N * 4));
    OO_CUDA(c, cudaMemcpyAsync(c->d_child, t->child, (size_t)N * 8 * 4, cudaMemcpyHostToDevice, stream));
    OO_CUDA(c, cudaMemcpyAsync(c->d_map_slot, t->map_slot, (size_t)N * 4, cudaMemcpyHostToDevice, stream));
    table_bytes += (uint64_t)N * 36;
    T.child = (const int32_t*)c->d_child;
    T.map_slot = (const int32_t*)c->d_map_slot;

    // ---- hop plan.  Stations: dense tables for every used depth <= Td and for Td = min(4, depth_eff) itself; each used
    // level deeper than Td must be within 3 depths of the previous station (else only the generic path is available).
    const uint32_t Td = std::min<uint32_t>(4, T.depth_eff);
    bool plan_ok = true;
    {
        uint32_t prev = Td;
        for (uint32_t l = 0; l < L; ++l) {
            const uint32_t d = t->level_depth[l];
            if (d <= Td) continue;
            if (d - prev > 3) plan_ok = false;
            prev = d;
        }
    }
    std::vector<std::vector<int32_t>> hop_host;    // kept alive until the stream sync below
    std::vector<int32_t> dense;
    if (plan_ok) {
        // node ids per depth and the integer cell coordinates of every node (by walking from the root)
        std::vector<uint32_t> cx(N), cy(N), cz(N);
        std::vector<std::vector<uint32_t>> by_depth(D + 1);
        cx[0] = cy[0] = cz[0] = 0;
        // parents precede children is NOT required by the ABI: do a BFS
        std::vector<uint32_t> queue;
        queue.reserve(N);
        queue.push_back(0);
        for (size_t h = 0; h < queue.size(); ++h) {
            const uint32_t i = queue[h];
            by_depth[t->depth[i]].push_back(i);
            for (int o = 0; o < 8; ++o) {
                const int32_t ch = t->child[(size_t)i * 8 + o];
                if (ch < 0) continue;
                cx[ch] = cx[i] * 2 + (o & 1); cy[ch] = cy[i] * 2 + ((o >> 1) & 1); cz[ch] = cz[i] * 2 + ((o >> 2) & 1);
                queue.push_back((uint32_t)ch);
            }
        }
        auto add_dense = [&](uint32_t d) -> uint32_t {
            const uint32_t off = (uint32_t)dense.size();
            dense.resize(off + (1u << (3 * d)), -1);
            for (uint32_t i : by_depth[d]) dense[off + ((cz[i] << (2 * d)) | (cy[i] << d) | cx[i])] = local[i];
            return off;
        };
        bool t_done = false;
        for (uint32_t l = 0; l < L; ++l) {
            LevelParams& lv = T.lv[l];
            if (lv.depth <= Td) {
                lv.dense = 1;
                lv.dense_off = add_dense(lv.depth);
                if (lv.depth == Td) { T.t_dense_off = lv.dense_off; t_done = true; }
            }
        }
        if (!t_done) T.t_dense_off = add_dense(Td);
        T.t_depth = Td;
        T.t_shift = T.depth_eff - Td;
        while (dense.size() % 4) dense.push_back(-1);
        T.dense_ints = (uint32_t)dense.size();
        OO_CUDA(c, cudaMalloc(&c->d_dense, dense.size() * 4));
        OO_CUDA(c, cudaMemcpyAsync(c->d_dense, dense.data(), dense.size() * 4, cudaMemcpyHostToDevice, stream));
        T.dense = (const int32_t*)c->d_dense;
        table_bytes += dense.size() * 4;
        // hop tables
        uint32_t prev_depth = Td;
        for (uint32_t l = 0; l < L; ++l) {
            LevelParams& lv = T.lv[l];
            if (lv.depth <= Td) continue;
            const uint32_t gdep = lv.depth - prev_depth;
            lv.dense = 0;
            lv.gap = gdep;
            // one row of 8^gap entries per local index at the previous station (a used level's local index is its
            // map_slot, which ranges over level_slots; an unused depth's is a running count over its nodes)
            size_t rows = std::max<size_t>(by_depth[prev_depth].size(), 1);
            const int pl = level_of_depth[prev_depth];
            if (pl >= 0) rows = std::max<size_t>(t->level_slots[pl], 1);
            if (((uint64_t)rows << (3 * gdep)) >= (1ull << 32))      // the kernels index a hop table with 32 bits
                return fail(c, OO_ERR_UNSUPPORTED, "level %u: a hop table of %llu entries (>= 2^32, 16 GB)", l, (unsigned long long)rows << (3 * gdep));
            hop_host.emplace_back(rows << (3 * gdep), -1);
            std::vector<int32_t>& tab = hop_host.back();
            const uint32_t m = (1u << gdep) - 1;
            // for every node at the previous station enumerate its descendants `gap` levels below
            std::vector<std::pair<uint32_t, uint32_t>> frontier, next;   // (node, ancestor local index)
            for (uint32_t a : by_depth[prev_depth]) frontier.emplace_back(a, (uint32_t)local[a]);
            for (uint32_t s = 0; s < gdep; ++s) {
                next.clear();
                for (auto& pr : frontier)
                    for (int o = 0; o < 8; ++o) {
                        const int32_t ch = t->child[(size_t)pr.first * 8 + o];
                        if (ch >= 0) next.emplace_back((uint32_t)ch, pr.second);
                    }
                frontier.swap(next);
            }
            for (auto& pr : frontier) {
                const uint32_t i = pr.first;
                const uint32_t idx = ((cz[i] & m) << (2 * gdep)) | ((cy[i] & m) << gdep) | (cx[i] & m);
                tab[((size_t)pr.second << (3 * gdep)) + idx] = local[i];
            }
            void* dptr = nullptr;
            OO_CUDA(c, cudaMalloc(&dptr, tab.size() * 4));
            c->d_hop.push_back(dptr);
            OO_CUDA(c, cudaMemcpyAsync(dptr, tab.data(), tab.size() * 4, cudaMemcpyHostToDevice, stream));
            lv.hop = (const int32_t*)dptr;
            table_bytes += tab.size() * 4;
            prev_depth = lv.depth;
        }
    }
    c->info.node_table_bytes = table_bytes;
    c->info.launches += (uint64_t)launches;
    c->info.tied_vertices = 0;
    if (d_changed) {
        unsigned long long h = 0;
        const cudaError_t e = cudaMemcpyAsync(&h, d_changed, sizeof h, cudaMemcpyDeviceToHost, stream);
        const cudaError_t e2 = e == cudaSuccess ? cudaStreamSynchronize(stream) : e;
        OO_CUDA(c, e2);
        c->info.tied_vertices = h;
    }
    OO_CUDA(c, cudaStreamSynchronize(stream));
    OO_CUDA(c, cudaGetLastError());
    c->T = T;
    c->plan_ok = plan_ok;
    c->have_tree = true;
    if (c->have_mlp) c->M.feat_dim = L * T.F;
    return OO_OK;
}

// The decoder weights in the UMMA K-major canonical layout (SWIZZLE_NONE): per layer chunk-major [K/8][N][8] halves; layer 0
// zero-padded to K1 = in_dim rounded up to 16, the output layer to N = 16 rows.
static std::vector<uint16_t> make_tc_image(uint32_t in_dim, uint32_t W, uint32_t n_hidden, uint32_t out_dim, const void* const* weights) {
    const uint32_t k1 = (in_dim + 15) & ~15u;
    std::vector<uint16_t> tc((size_t)k1 * W + (size_t)(n_hidden - 1) * W * W + (size_t)W * 16, 0);
    auto put = [&](size_t base, uint32_t N, uint32_t n, uint32_t k, uint16_t v) { tc[base + ((size_t)(k / 8) * N + n) * 8 + (k % 8)] = v; };
    const uint16_t* w0 = (const uint16_t*)weights[0];
    for (uint32_t o = 0; o < W; ++o)
        for (uint32_t i = 0; i < in_dim; ++i) put(0, W, o, i, w0[(size_t)o * in_dim + i]);
    size_t base = (size_t)k1 * W;
    for (uint32_t k = 1; k < n_hidden; ++k) {
        const uint16_t* w = (const uint16_t*)weights[k];
        for (uint32_t o = 0; o < W; ++o)
            for (uint32_t i = 0; i < W; ++i) put(base, W, o, i, w[(size_t)o * W + i]);
        base += (size_t)W * W;
    }
    const uint16_t* wl = (const uint16_t*)weights[n_hidden];
    for (uint32_t o = 0; o < out_dim; ++o)
        for (uint32_t i = 0; i < W; ++i) put(base, 16, o, i, wl[(size_t)o * W + i]);
    return tc;
}

// ---------------------------------------------------------------------------------------------------------------------
// oo_upload_mlp
// ---------------------------------------------------------------------------------------------------------------------
extern "C" OO_API oo_status oo_upload_mlp(oo_ctx* c, const oo_mlp_desc* m, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!m || !m->weights) return fail(c, OO_ERR_INVALID_ARG, "mlp or mlp.weights is NULL");
    if (m->width != 64 && m->width != 128) return fail(c, OO_ERR_UNSUPPORTED, "hidden width %u: only 64 and 128 are implemented", m->width);
    const uint32_t W = m->width;
    if (m->n_hidden < 1 || m->n_hidden > OO_MAX_HIDDEN) return fail(c, OO_ERR_INVALID_ARG, "n_hidden %u outside 1..%d", m->n_hidden, OO_MAX_HIDDEN);
    if (m->out_dim < 1 || m->out_dim > 8) return fail(c, OO_ERR_INVALID_ARG, "out_dim %u outside 1..8", m->out_dim);
    // widest input the ABI describes: L*F <= OO_MAX_LEVELS*32 features + 9 attributes (OO_ATTRS_PAPER) + OO_MAX_EXTRA extras
    if (m->in_dim < 7 || m->in_dim > OO_MAX_LEVELS * 32 + 9 + OO_MAX_EXTRA) return fail(c, OO_ERR_INVALID_ARG, "in_dim %u outside 7..%d", m->in_dim, OO_MAX_LEVELS * 32 + 9 + OO_MAX_EXTRA);
    if (m->out_act != OO_ACT_NONE && m->out_act != OO_ACT_EXP) return fail(c, OO_ERR_INVALID_ARG, "unknown out_act");
    for (uint32_t k = 0; k <= m->n_hidden; ++k)
        if (!m->weights[k]) return fail(c, OO_ERR_INVALID_ARG, "weights[%u] is NULL", k);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g(c->device);
    // weights_on_device: the matrices are DEVICE buffers (e.g. a trainer's parameters): bring them to the host first, the
    // padded images are built there either way (a few tens of KB, once per upload)
    std::vector<std::vector<uint16_t>> staged;
    std::vector<const void*> host_w(m->n_hidden + 1);
    for (uint32_t k = 0; k <= m->n_hidden; ++k) host_w[k] = m->weights[k];
    if (m->weights_on_device) {
        staged.resize(m->n_hidden + 1);
        for (uint32_t k = 0; k <= m->n_hidden; ++k) {
            const size_t rows = k == m->n_hidden ? m->out_dim : W, cols = k == 0 ? m->in_dim : W;
            staged[k].resize(rows * cols);
            OO_CUDA(c, cudaMemcpyAsync(staged[k].data(), m->weights[k], rows * cols * 2, cudaMemcpyDeviceToHost, stream));
            host_w[k] = staged[k].data();
        }
        OO_CUDA(c, cudaStreamSynchronize(stream));
    }
    const void* const* weights = host_w.data();
    const uint32_t k1 = (m->in_dim + 15) & ~15u;
    const uint32_t s0 = k1 + 8, s1 = 72;
    const size_t halves = (size_t)64 * s0 + (size_t)(m->n_hidden - 1) * 64 * s1 + (size_t)16 * s1;
    std::vector<uint16_t> img(halves, 0);     // the mma.sync image (width 64 only; left zero otherwise and never used)
    const uint16_t* w0 = (const uint16_t*)weights[0];
    if (W == 64)
    for (uint32_t o = 0; o < 64; ++o)
        for (uint32_t i = 0; i < m->in_dim; ++i) img[(size_t)o * s0 + i] = w0[(size_t)o * m->in_dim + i];
    size_t off = (size_t)64 * s0;
    for (uint32_t k = 1; W == 64 && k < m->n_hidden; ++k) {
        const uint16_t* w = (const uint16_t*)weights[k];
        for (uint32_t o = 0; o < 64; ++o)
            for (uint32_t i = 0; i < 64; ++i) img[off + (size_t)o * s1 + i] = w[(size_t)o * 64 + i];
        off += (size_t)64 * s1;
    }
    const uint16_t* wl = (const uint16_t*)weights[m->n_hidden];
    for (uint32_t o = 0; W == 64 && o < m->out_dim; ++o)
        for (uint32_t i = 0; i < 64; ++i) img[off + (size_t)o * s1 + i] = wl[(size_t)o * 64 + i];
    const std::vector<uint16_t> tc = make_tc_image(m->in_dim, W, m->n_hidden, m->out_dim, weights);
    const size_t tc_halves = tc.size();
    free_dev(c->d_image);
    free_dev(c->d_image_tc);
    c->have_mlp = false;
    OO_CUDA(c, cudaMalloc(&c->d_image, halves * 2));
    OO_CUDA(c, cudaMemcpyAsync(c->d_image, img.data(), halves * 2, cudaMemcpyHostToDevice, stream));
    OO_CUDA(c, cudaMalloc(&c->d_image_tc, tc_halves * 2));
    OO_CUDA(c, cudaMemcpyAsync(c->d_image_tc, tc.data(), tc_halves * 2, cudaMemcpyHostToDevice, stream));
    OO_CUDA(c, cudaStreamSynchronize(stream));
    MlpParams M{};
    M.image = (const uint16_t*)c->d_image;
    M.image_bytes = (uint32_t)(halves * 2);
    M.in_dim = m->in_dim; M.k1 = k1; M.n_hidden = m->n_hidden; M.out_dim = m->out_dim; M.out_act = (uint32_t)m->out_act;
    M.feat_dim = c->have_tree ? c->T.n_levels * c->T.F : 0;
    M.image_tc = (const uint16_t*)c->d_image_tc;
    M.image_tc_bytes = (uint32_t)(tc_halves * 2);
    M.width = W;
    c->M = M;
    c->have_mlp = true;
    return OO_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// oo_upload_disparity
// ---------------------------------------------------------------------------------------------------------------------
extern "C" OO_API oo_status oo_upload_disparity(oo_ctx* c, const oo_disparity_desc* d, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!d || !d->res || !d->tables || !d->weights) return fail(c, OO_ERR_INVALID_ARG, "disparity descriptor or one of its arrays is NULL");
    if (d->n_levels < 1 || d->n_levels > OO_MAX_GRID_LEVELS) return fail(c, OO_ERR_INVALID_ARG, "n_levels %u outside 1..%d", d->n_levels, OO_MAX_GRID_LEVELS);
    if (d->n_features != 2) return fail(c, OO_ERR_UNSUPPORTED, "n_features %u: only 2 (one 32-bit entry) is implemented", d->n_features);
    if (d->hash_log2 < 4 || d->hash_log2 > 28) return fail(c, OO_ERR_INVALID_ARG, "hash_log2 %u outside 4..28", d->hash_log2);
    if (d->n_hidden < 1 || d->n_hidden > OO_MAX_HIDDEN) return fail(c, OO_ERR_INVALID_ARG, "n_hidden %u outside 1..%d", d->n_hidden, OO_MAX_HIDDEN);
    const uint64_t t_max = 1ull << d->hash_log2;
    std::vector<uint64_t> entries(d->n_levels), offset(d->n_levels);
    uint64_t total = 0;
    for (uint32_t g = 0; g < d->n_levels; ++g) {
        const uint64_t N = d->res[g];
        if (N < 1 || N > (1u << 20)) return fail(c, OO_ERR_INVALID_ARG, "res[%u] = %llu outside 1..2^20", g, (unsigned long long)N);
        if (!d->tables[g]) return fail(c, OO_ERR_INVALID_ARG, "tables[%u] is NULL", g);
        const uint64_t dense = (N + 1) * (N + 1) * (N + 1);
        entries[g] = dense <= t_max ? dense : t_max;
        offset[g] = total;
        total += entries[g];
    }
    for (uint32_t k = 0; k <= d->n_hidden; ++k)
        if (!d->weights[k]) return fail(c, OO_ERR_INVALID_ARG, "weights[%u] is NULL", k);
    const uint32_t in_dim = 2 * d->n_levels + 3;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g(c->device);
    const std::vector<uint16_t> tc = make_tc_image(in_dim, 64, d->n_hidden, 1, d->weights);
    free_dev(c->d_grid);
    free_dev(c->d_disp_image);
    c->have_disp = false;
    OO_CUDA(c, cudaMalloc(&c->d_grid, total * 4));
    OO_CUDA(c, cudaMalloc(&c->d_disp_image, tc.size() * 2));
    GridParams G{};
    G.n_levels = d->n_levels;
    for (uint32_t l = 0; l < d->n_levels; ++l) {
        OO_CUDA(c, cudaMemcpyAsync((uint32_t*)c->d_grid + offset[l], d->tables[l], entries[l] * 4, cudaMemcpyHostToDevice, stream));
        GridLevel& lv = G.lv[l];
        lv.table = (const uint32_t*)c->d_grid + offset[l];
        lv.scale = (float)d->res[l];
        lv.n_max = d->res[l] - 1;
        lv.stride = d->res[l] + 1;
        lv.mask = entries[l] == t_max && (uint64_t)(d->res[l] + 1) * (d->res[l] + 1) * (d->res[l] + 1) > t_max ? (uint32_t)(t_max - 1) : 0u;
    }
    {
        uint32_t nd = 0;
        while (nd < G.n_levels && !G.lv[nd].mask) ++nd;
        G.n_dense = nd;
        for (uint32_t l = nd; l < G.n_levels; ++l)
            if (!G.lv[l].mask) G.n_dense = G.n_levels + 1;
    }
    OO_CUDA(c, cudaMemcpyAsync(c->d_disp_image, tc.data(), tc.size() * 2, cudaMemcpyHostToDevice, stream));
    OO_CUDA(c, cudaStreamSynchronize(stream));
    MlpParams M{};
    M.in_dim = in_dim; M.k1 = (in_dim + 15) & ~15u; M.n_hidden = d->n_hidden; M.out_dim = 1; M.out_act = (uint32_t)OO_ACT_EXP;
    M.image_tc = (const uint16_t*)c->d_disp_image;
    M.image_tc_bytes = (uint32_t)(tc.size() * 2);
    M.width = 64;
    c->G = G;
    c->MD = M;
    c->have_disp = true;
    return OO_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// scratch
// ---------------------------------------------------------------------------------------------------------------------
// Bytes of feature scratch OO_PATH_GENERIC / OO_PATH_UNFUSED need for n queries of the uploaded tree (0 without a tree)
static uint64_t feat_bytes_for(const oo_ctx* c, uint64_t n) {
    return c->have_tree ? n * (uint64_t)c->T.n_levels * c->T.texel_bytes : 0;
}

extern "C" OO_API oo_status oo_reserve(oo_ctx* c, uint64_t n) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (c->sticky != cudaSuccess) return fail(c, OO_ERR_CUDA, "earlier CUDA failure: %s", cudaGetErrorString(c->sticky));
    DeviceGuard g(c->device);
    // feature rows of the unfused paths depend on the uploaded tree: (re)sized here even when the row count is unchanged,
    // so that "oo_upload_tree, then oo_reserve" is always enough and no hot call has to allocate
    const uint64_t rows = std::max(n, c->reserved);
    const uint64_t fb = feat_bytes_for(c, rows);
    if (fb > c->feat_bytes) {
        free_dev(c->d_feat);
        c->feat_bytes = 0;
        OO_CUDA(c, cudaMalloc(&c->d_feat, fb));
        c->feat_bytes = fb;
    }
    if (n <= c->reserved) return OO_OK;
    void* keep_feat = c->d_feat;
    const uint64_t keep_fb = c->feat_bytes;
    c->d_feat = nullptr;
    free_scratch(c);
    c->d_feat = keep_feat;
    c->feat_bytes = keep_fb;
    OO_CUDA(c, cudaMalloc((void**)&c->d_keys_a, n * 4));
    OO_CUDA(c, cudaMalloc((void**)&c->d_keys_b, n * 4));
    OO_CUDA(c, cudaMalloc((void**)&c->d_idx_a, n * 4));
    OO_CUDA(c, cudaMalloc((void**)&c->d_hist, morton_sort_hist_ints(n) * 4));
    OO_CUDA(c, cudaMalloc((void**)&c->d_qx, n * 12));
    OO_CUDA(c, cudaMalloc((void**)&c->d_qn, n * 12));
    OO_CUDA(c, cudaMalloc((void**)&c->d_qw, n * 12));
    OO_CUDA(c, cudaMalloc((void**)&c->d_qe, n * 4 * OO_MAX_EXTRA));
    OO_CUDA(c, cudaMalloc((void**)&c->d_rgb, n * 4 * 8));
    OO_CUDA(c, cudaMalloc((void**)&c->d_qd, n * 4));
    // OO_PRESORT_BIN: the binned copy of the queries, both index maps, the binned RGB and d^
    OO_CUDA(c, cudaMalloc((void**)&c->d_bx, n * 12));
    OO_CUDA(c, cudaMalloc((void**)&c->d_bn, n * 12));
    OO_CUDA(c, cudaMalloc((void**)&c->d_bw, n * 12));
    OO_CUDA(c, cudaMalloc((void**)&c->d_be, n * 4 * OO_MAX_EXTRA));
    OO_CUDA(c, cudaMalloc((void**)&c->d_binv, n * 4));
    OO_CUDA(c, cudaMalloc((void**)&c->d_bidx, n * 4));
    OO_CUDA(c, cudaMalloc((void**)&c->d_brgb, n * 4 * 8));
    OO_CUDA(c, cudaMalloc((void**)&c->d_bdisp, n * 4));
    OO_CUDA(c, cudaMalloc((void**)&c->d_btot, 1024 * 4));
    OO_CUDA(c, cudaMemset(c->d_btot, 0, 1024 * 4));
    c->reserved = n;
    return OO_OK;
}

// Hot calls never allocate: the scratch they need must have been reserved.
static oo_status need_feat(oo_ctx* c, uint64_t bytes) {
    if (bytes <= c->feat_bytes) return OO_OK;
    return fail(c, OO_ERR_NOT_READY, "OO_PATH_GENERIC / OO_PATH_UNFUSED keep the feature rows in scratch: call oo_reserve(n) after oo_upload_tree (need %llu bytes, have %llu)",
                (unsigned long long)bytes, (unsigned long long)c->feat_bytes);
}
static oo_status need_bin(oo_ctx* c, uint64_t n) {
    if (n <= c->reserved) return OO_OK;
    return fail(c, OO_ERR_NOT_READY, "OO_PRESORT_BIN: call oo_reserve(%llu) first", (unsigned long long)n);
}

// a1' for oo_query: one counting pass on the top Morton bits moves the queries (and a caller-supplied d^) into the binned
// scratch; *qb then describes the binned copy.  The chosen kernel runs over it into c->d_brgb and unbin restores the order.
// OO_PRESORT_AUTO: fold the newest coherence sample the kernels have left into the decision.  Slots carry the sequence number of
// the call that wrote them; the newest call present wins (a call still running contributes the blocks that have finished).
// Hysteresis: on above 12 distinct cells per 32 queries, off below 6 (screen-order frames measure 1-3, random surface samples ~30).
static void update_coherence(oo_ctx* c) {
    if (!c->ev_stat) return;
    const uint32_t mask = (1u << kStatSeqBits) - 1u;
    uint32_t best_age = ~0u;
    uint64_t sum = 0, cnt = 0;
    for (uint32_t k = 0; k < kStatSlots; ++k) {
        const unsigned long long v = ((volatile unsigned long long*)c->h_stat)[k];
        const uint32_t n = (uint32_t)(v >> 32) & ((1u << kStatCntBits) - 1u);
        if (!n) continue;
        const uint32_t age = (c->stat_seq - (uint32_t)(v >> 44)) & mask;
        if (age < best_age) { best_age = age; sum = cnt = 0; }
        if (age == best_age) { sum += (uint32_t)v; cnt += n; }
    }
    if (cnt < 16) return;                     // too few warps sampled to say anything
    c->coherence = (float)sum / (float)cnt;
    c->auto_on = c->coherence > (c->auto_on ? 6.0f : 12.0f);
}
// Does this call sample?  (Only under AUTO; the kernel that sees the caller's order gets the pointer.)
static void arm_sampling(oo_ctx* c, QueryParams& Q) {
    if (c->presort != OO_PRESORT_AUTO || !c->ev_stat || Q.perm) return;
    c->stat_seq = (c->stat_seq + 1) & ((1u << kStatSeqBits) - 1u);
    Q.stat = c->d_stat;
    Q.stat_seq = c->stat_seq;
    c->armed = true;
}
// After the kernels of a sampling call have been enqueued on the caller's stream: the side stream waits for them and copies the
// sample array to the host.  Nothing is added to the caller's stream but an event record; failures only lose the sample.
// While the caller's stream is being CAPTURED into a CUDA graph the copy is left out: waiting on an event recorded in a capturing
// stream would pull the side stream into the capture, where it never rejoins (cudaStreamEndCapture then fails with
// cudaErrorStreamCaptureUnjoined).  The kernels still write their samples to the device array, which is harmless; a replayed
// graph repeats the decision that was current when it was captured.
static void collect_samples(oo_ctx* c, cudaStream_t stream) {
    if (!c->armed) return;
    c->armed = false;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(stream, &cap) != cudaSuccess) { (void)cudaGetLastError(); return; }
    if (cap != cudaStreamCaptureStatusNone) return;
    if (cudaEventRecord(c->ev_stat, stream) != cudaSuccess || cudaStreamWaitEvent(c->s_stat, c->ev_stat, 0) != cudaSuccess ||
        cudaMemcpyAsync(c->h_stat, c->d_stat, kStatSlots * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->s_stat) != cudaSuccess)
        (void)cudaGetLastError();
}
// Will this batch's taps miss the caches?  Binned queries do by construction (they are incoherent or they would not have been binned);
// otherwise, under OO_PRESORT_AUTO (the only mode that samples), the latest coherence sample decides.  Chooses between the two encode kernels.
static bool cache_cold(oo_ctx* c, bool binned) {
    if (binned) return true;
    if (c->presort != OO_PRESORT_AUTO) return false;
    update_coherence(c);                   // (batches below the binning threshold have not been through bin_wanted's update)
    return c->coherence > 12.0f;
}
static bool bin_wanted(oo_ctx* c, const oo_queries* q) {
    if (q->perm || q->n < c->bin_min) return false;
    if (c->presort == OO_PRESORT_BIN) return true;
    if (c->presort != OO_PRESORT_AUTO) return false;
    update_coherence(c);
    return c->auto_on && q->n <= c->reserved;      // AUTO never fails a call for missing scratch: it proceeds unsorted
}
static oo_status bin_for_query(oo_ctx* c, const oo_queries* q, oo_queries* qb, cudaStream_t stream, bool want_idx = false) {
    if (oo_status st = need_bin(c, q->n)) return st;
    QueryParams Qs = make_qp(q);
    arm_sampling(c, Qs);                     // binned call: the histogram kernel is the one that sees the caller's order
    const int k = launch_bin_queries(Qs, c->d_keys_a, c->d_hist, c->d_btot, c->d_bx, c->d_bn, c->d_bw, c->d_be, c->d_binv,
                                     want_idx ? c->d_bidx : nullptr, q->disparity ? c->d_bdisp : nullptr, stream);
    if (k < 0) return launch_failed(c, k, "bin pass");
    count(c, k);
    *qb = *q;
    qb->x = c->d_bx; qb->nrm = c->d_bn; qb->wo = c->d_bw;
    qb->extra = q->n_extra && q->extra ? c->d_be : nullptr;
    qb->disparity = q->disparity ? c->d_bdisp : nullptr;
    return OO_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// oo_sort_queries
// ---------------------------------------------------------------------------------------------------------------------
extern "C" OO_API oo_status oo_sort_queries(oo_ctx* c, const oo_queries* q, uint32_t* d_perm_out, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!q || (q->n && (!q->x || !d_perm_out))) return fail(c, OO_ERR_INVALID_ARG, "NULL argument");
    if (q->n >= (1ull << 32)) return fail(c, OO_ERR_UNSUPPORTED, "more than 2^32-1 queries per call");
    if (q->n > c->reserved) return fail(c, OO_ERR_NOT_READY, "call oo_reserve(%llu) first", (unsigned long long)q->n);
    if (oo_status st = check_before(c)) return st;
    DeviceGuard g(c->device);
    const int k = launch_morton_sort(q->x, q->n, c->d_keys_a, c->d_keys_b, c->d_idx_a, d_perm_out, c->d_hist, (cudaStream_t)cuda_stream);
    if (k < 0) return launch_failed(c, k, "Morton sort");
    count(c, k);
    return check_after(c);
}

// ---------------------------------------------------------------------------------------------------------------------
// oo_encode / oo_query
// ---------------------------------------------------------------------------------------------------------------------
static oo_path resolve_encode_path(oo_ctx* c) {
    const bool fast = c->plan_ok && fast_shape_supported(c->T.n_levels, c->T.F, c->T.f32 != 0);
    if (c->path == OO_PATH_GENERIC) return OO_PATH_GENERIC;
    if (c->path == OO_PATH_AUTO) return fast ? OO_PATH_UNFUSED : OO_PATH_GENERIC;
    return fast ? OO_PATH_UNFUSED : (oo_path)-1;
}

extern "C" OO_API oo_status oo_encode(oo_ctx* c, const oo_queries* q, void* d_features, int32_t* d_slot, int16_t* d_texel,
                               void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!c->have_tree) return fail(c, OO_ERR_NOT_READY, "no tree uploaded");
    if (c->T.vertex) return fail(c, OO_ERR_UNSUPPORTED, "oo_encode reads texel maps; use oo_encode_full for vertex maps");
    if (oo_status st = check_queries(c, q, false)) return st;
    if (oo_status st = check_before(c)) return st;
    if (q->n == 0) return OO_OK;
    DeviceGuard g(c->device);
    const oo_path p = resolve_encode_path(c);
    if ((int)p < 0) return fail(c, OO_ERR_UNSUPPORTED, "no specialised kernel for L=%u F=%u (or the tree has no hop plan); use OO_PATH_GENERIC/AUTO", c->T.n_levels, c->T.F);
    QueryParams Q = make_qp(q);
    EncodeOut O{d_features, d_slot, d_texel};
    c->info.presorted_last_encode = 0;
    if (p == OO_PATH_UNFUSED && bin_wanted(c, q)) {
        // a1': x and wo move into Morton bins; the encode kernel reads them in order and stores every row at its query's index
        if (oo_status st = need_bin(c, q->n)) return st;
        Q.nrm = nullptr; Q.extra = nullptr; Q.n_extra = 0;
        arm_sampling(c, Q);
        const int k = launch_bin_queries(Q, c->d_keys_a, c->d_hist, c->d_btot, c->d_bx, c->d_bn, c->d_bw, c->d_be, c->d_binv, c->d_bidx, nullptr, (cudaStream_t)cuda_stream);
        if (k < 0) return launch_failed(c, k, "bin pass");
        count(c, k);
        Q.x = c->d_bx; Q.wo = c->d_bw; Q.out_idx = c->d_bidx;
        Q.stat = nullptr;
        c->info.presorted_last_encode = 1;
    } else if (p == OO_PATH_UNFUSED) {
        arm_sampling(c, Q);
    }
    bool pipelined = false;
    int n = p == OO_PATH_GENERIC ? launch_encode_generic(c->T, Q, O, c->tree_max_depth, (cudaStream_t)cuda_stream)
                                 : launch_encode_fast(c->T, Q, O, c->n_sms, (cudaStream_t)cuda_stream, cache_cold(c, c->info.presorted_last_encode != 0), &pipelined);
    if (n < 0) return launch_failed(c, n, "encode kernel");
    count(c, n);
    c->info.path_last_encode = (uint32_t)p;
    c->info.encode_pipelined_last = pipelined ? 1u : 0u;
    collect_samples(c, (cudaStream_t)cuda_stream);
    return check_after(c);
}

// the full-query kernels are needed as soon as anything differs from the hot path
static bool needs_full(const oo_ctx* c) {
    return c->mode.tri8 || c->mode.lookup || c->mode.attrs_paper || c->T.vertex || (c->have_mlp && c->M.width != 64);
}

static oo_status check_full(oo_ctx* c, const oo_queries* q) {
    if (!c->plan_ok) return fail(c, OO_ERR_UNSUPPORTED, "the full query needs the hop-table descent (used depths at most 3 apart below depth 4)");
    if (c->mode.lookup != OO_LOOKUP_WO && q->n && !q->nrm) return fail(c, OO_ERR_INVALID_ARG, "queries.nrm is NULL (mirror direction)");
    if (c->mode.lookup == OO_LOOKUP_SHIFTED && q->n && !q->disparity) {
        if (!c->have_disp) return fail(c, OO_ERR_INVALID_ARG, "queries.disparity is NULL (OO_LOOKUP_SHIFTED) and no disparity predictor is uploaded");
        if (q->n > c->reserved) return fail(c, OO_ERR_NOT_READY, "predicting the disparity needs scratch: call oo_reserve(%llu) first", (unsigned long long)q->n);
    }
    return OO_OK;
}

// Eq. 7: d^ = g_psi(x, w_r) for every query, into d_out (DEVICE [n]); optionally the hash-grid features.
static oo_status predict_disparity(oo_ctx* c, const oo_queries* q, float* d_out, float* d_features, cudaStream_t stream) {
    if (!c->have_disp) return fail(c, OO_ERR_NOT_READY, "no disparity predictor uploaded");
    if (oo_status st = check_queries(c, q, true)) return st;
    if (q->n && !d_out) return fail(c, OO_ERR_INVALID_ARG, "disparity output is NULL");
    if (oo_status st = check_before(c)) return st;
    if (q->n == 0) return OO_OK;
    const int n = launch_disparity(c->G, c->MD, make_qp(q), d_out, d_features, c->n_sms, stream);
    if (n < 0) return launch_failed(c, n, "disparity kernel");
    count(c, n);
    return check_after(c);
}

// OO_LOOKUP_SHIFTED without a caller-supplied d^: run the predictor into the context's scratch and point the queries at it.
static oo_status fill_disparity(oo_ctx* c, oo_queries* q, cudaStream_t stream) {
    if (c->mode.lookup != OO_LOOKUP_SHIFTED || q->disparity || q->n == 0) return OO_OK;
    if (oo_status st = predict_disparity(c, q, c->d_qd, nullptr, stream)) return st;
    q->disparity = c->d_qd;
    return OO_OK;
}

extern "C" OO_API oo_status oo_predict_disparity(oo_ctx* c, const oo_queries* q, float* d_disparity, float* d_features, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    DeviceGuard g(c->device);
    return predict_disparity(c, q, d_disparity, d_features, (cudaStream_t)cuda_stream);
}

extern "C" OO_API oo_status oo_encode_full(oo_ctx* c, const oo_queries* q, float* d_features, int32_t* d_slot, int16_t* d_cell,
                                    void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!c->have_tree) return fail(c, OO_ERR_NOT_READY, "no tree uploaded");
    if (oo_status st = check_queries(c, q, false)) return st;
    if (oo_status st = check_full(c, q)) return st;
    if (oo_status st = check_before(c)) return st;
    if (q->n == 0) return OO_OK;
    DeviceGuard g(c->device);
    oo_queries qd = *q;
    if (oo_status st = fill_disparity(c, &qd, (cudaStream_t)cuda_stream)) return st;
    q = &qd;
    const int n = launch_encode_full(c->T, make_qp(q), c->mode, d_features, d_slot, d_cell, c->n_sms, (cudaStream_t)cuda_stream);
    if (n < 0) return launch_failed(c, n, "full-query encode kernel (F, dtype)");
    count(c, n);
    c->info.path_last_encode = (uint32_t)OO_PATH_FULL;
    return check_after(c);
}

// Debug outputs of oo_query_debug (null for oo_query)
struct DebugOut {
    int32_t* slot = nullptr;
    int16_t* index = nullptr;
    bool on() const { return slot || index; }
};

static const char* path_name(oo_path p) {
    switch (p) {
        case OO_PATH_GENERIC: return "OO_PATH_GENERIC";
        case OO_PATH_UNFUSED: return "OO_PATH_UNFUSED";
        case OO_PATH_FUSED_MMA: return "OO_PATH_FUSED_MMA";
        case OO_PATH_FUSED_TC: return "OO_PATH_FUSED_TC";
        case OO_PATH_FUSED_TC_TMEM: return "OO_PATH_FUSED_TC_TMEM";
        case OO_PATH_FULL: return "OO_PATH_FULL";
        default: return "OO_PATH_AUTO";
    }
}

static oo_status query_device(oo_ctx* c, const oo_queries* q, float* d_rgb, cudaStream_t stream, const DebugOut& dbg = DebugOut()) {
    if (!c->have_tree) return fail(c, OO_ERR_NOT_READY, "no tree uploaded");
    if (!c->have_mlp) return fail(c, OO_ERR_NOT_READY, "no MLP uploaded");
    if (oo_status st = check_queries(c, q, true)) return st;
    if (q->n && !d_rgb) return fail(c, OO_ERR_INVALID_ARG, "rgb is NULL");
    const uint32_t feat = c->T.n_levels * c->T.F;
    const uint32_t n_attr = c->mode.attrs_paper ? 9u : 6u;
    if (c->M.in_dim != feat + n_attr + q->n_extra)
        return fail(c, OO_ERR_NOT_READY, "MLP in_dim %u != L*F + %u + n_extra = %u", c->M.in_dim, n_attr, feat + n_attr + q->n_extra);
    const bool full = needs_full(c);
    if (full) {
        if (oo_status st = check_full(c, q)) return st;
        if (c->path != OO_PATH_AUTO) return fail(c, OO_ERR_UNSUPPORTED, "the full query has one kernel; oo_set_path(OO_PATH_AUTO)");
    }
    if (oo_status st = check_before(c)) return st;
    if (q->n == 0) return OO_OK;
    c->M.feat_dim = feat;
    // ---- a1 inside the query: bin the queries first (the predictor's hash-grid gathers profit from the order too)
    oo_queries qd = *q;
    float* out = d_rgb;
    c->info.presorted_last_query = 0;
    if (bin_wanted(c, q)) {
        if (oo_status st = bin_for_query(c, q, &qd, stream, dbg.on())) return st;
        out = c->d_brgb;
        c->info.presorted_last_query = 1;
    }
    QueryParams Q;
    int n = 0;
    oo_path p = c->path;
    if (full) {
        if (oo_status st = fill_disparity(c, &qd, stream)) return st;
        Q = make_qp(&qd);
        Q.dbg_slot = dbg.slot; Q.dbg_texel = dbg.index;
        if (c->info.presorted_last_query && dbg.on()) Q.out_idx = c->d_bidx;
        if (!c->info.presorted_last_query) arm_sampling(c, Q);
        if (dbg.on())
            n = c->M.width == 64 ? launch_fused_full_w64_dbg(c->T, c->M, Q, c->mode, out, c->n_sms, stream)
                                 : launch_fused_full_w128_dbg(c->T, c->M, Q, c->mode, out, c->n_sms, stream);
        else
            n = c->M.width == 64 ? launch_fused_full_w64(c->T, c->M, Q, c->mode, out, c->n_sms, stream)
                                 : launch_fused_full_w128(c->T, c->M, Q, c->mode, out, c->n_sms, stream);
        if (n < 0) return launch_failed(c, n, "full-query kernel (F, dtype, in_dim <= 128, out_dim <= 4)");
        p = OO_PATH_FULL;
    } else {
        const bool fast = c->plan_ok && fast_shape_supported(c->T.n_levels, c->T.F, c->T.f32 != 0);
        if (p == OO_PATH_AUTO) p = !fast ? OO_PATH_GENERIC : OO_PATH_FUSED_TC_TMEM;
        if (p != OO_PATH_GENERIC && !fast)
            return fail(c, OO_ERR_UNSUPPORTED, "no specialised kernel for L=%u F=%u (or the tree has no hop plan); use OO_PATH_GENERIC/AUTO", c->T.n_levels, c->T.F);
        Q = make_qp(&qd);
        Q.dbg_slot = dbg.slot; Q.dbg_texel = dbg.index;
        if (c->info.presorted_last_query && dbg.on()) Q.out_idx = c->d_bidx;
        if (!c->info.presorted_last_query) arm_sampling(c, Q);
        // OO_PATH_AUTO walks down the chain until a kernel exists for the shape: activations in tensor memory -> A tile in
        // shared memory -> mma.sync -> features through HBM.  An explicit path runs that kernel or fails.
        const bool walk = c->path == OO_PATH_AUTO;
        n = -1;
        if (p == OO_PATH_FUSED_TC_TMEM) {
            n = dbg.on() ? launch_fused_tm_dbg(c->T, c->M, Q, out, c->n_sms, stream) : launch_fused_tm(c->T, c->M, Q, out, c->n_sms, stream);
            if (n == -1 && walk) p = OO_PATH_FUSED_TC;
        }
        if (n == -1 && p == OO_PATH_FUSED_TC) {
            n = launch_fused_tc(c->T, c->M, Q, out, c->n_sms, stream, dbg.on());
            if (n == -1 && walk) p = OO_PATH_FUSED_MMA;
        }
        if (n == -1 && p == OO_PATH_FUSED_MMA) {
            n = launch_fused_mma(c->T, c->M, Q, out, c->n_sms, stream, dbg.on());
            if (n == -1 && walk) p = OO_PATH_UNFUSED;
        }
        if (n == -1 && (p == OO_PATH_GENERIC || p == OO_PATH_UNFUSED)) {
            const uint64_t bytes = q->n * (uint64_t)c->T.n_levels * c->T.texel_bytes;
            if (oo_status st = need_feat(c, bytes)) return st;
            // the encode kernels are their own debug instances: they take the index outputs as they are
            QueryParams Qe = Q;
            if (c->info.presorted_last_query) Qe.out_idx = nullptr;     // features stay in processing order for the MLP kernel ...
            EncodeOut O{c->d_feat, nullptr, nullptr};
            if (dbg.on() && !c->info.presorted_last_query) { O.slot = dbg.slot; O.texel = dbg.index; }
            n = p == OO_PATH_GENERIC ? launch_encode_generic(c->T, Qe, O, c->tree_max_depth, stream) : launch_encode_fast(c->T, Qe, O, c->n_sms, stream, cache_cold(c, c->info.presorted_last_query != 0));
            if (n < 0) return launch_failed(c, n, "encode kernel");
            count(c, n);
            if (dbg.on() && c->info.presorted_last_query) {             // ... so binned debug rows take a second, index-only pass
                QueryParams Qi = Q;
                Qi.out_idx = c->d_bidx;
                EncodeOut Oi{nullptr, dbg.slot, dbg.index};
                const int k = p == OO_PATH_GENERIC ? launch_encode_generic(c->T, Qi, Oi, c->tree_max_depth, stream) : launch_encode_fast(c->T, Qi, Oi, c->n_sms, stream, true);
                if (k < 0) return launch_failed(c, k, "encode kernel");
                count(c, k);
            }
            n = launch_mlp_rows(c->T, c->M, Qe, c->d_feat, out, c->n_sms, stream);
        }
        if (n < 0) return launch_failed(c, n, path_name(p));
        if (walk && p != OO_PATH_FUSED_TC_TMEM) {
            char buf[256];
            snprintf(buf, sizeof buf, "OO_PATH_AUTO resolved to %s for L=%u F=%u %s, in_dim %u, out_dim %u%s", path_name(p), c->T.n_levels, c->T.F,
                     c->T.f32 ? "fp32" : "fp16", c->M.in_dim, c->M.out_dim, c->plan_ok ? "" : " (the tree has no hop plan)");
            c->note = buf;
        } else {
            c->note.clear();
        }
    }
    count(c, n);
    if (c->info.presorted_last_query) count(c, launch_unbin(c->d_brgb, c->d_binv, q->n, c->M.out_dim, d_rgb, c->n_sms, stream));
    c->info.path_last_query = (uint32_t)p;
    collect_samples(c, stream);
    return check_after(c);
}

extern "C" OO_API oo_status oo_query(oo_ctx* c, const oo_queries* q, float* d_rgb, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    DeviceGuard g(c->device);
    return query_device(c, q, d_rgb, (cudaStream_t)cuda_stream);
}

extern "C" OO_API oo_status oo_query_debug(oo_ctx* c, const oo_queries* q, float* d_rgb, int32_t* d_slot, int16_t* d_index, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    DeviceGuard g(c->device);
    DebugOut dbg;
    dbg.slot = d_slot;
    dbg.index = d_index;
    return query_device(c, q, d_rgb, (cudaStream_t)cuda_stream, dbg);
}

extern "C" OO_API oo_status oo_set_host_chunks(oo_ctx* c, uint32_t n_chunks) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (n_chunks > (uint32_t)oo_ctx::kMaxChunks) return fail(c, OO_ERR_INVALID_ARG, "n_chunks %u outside 0..%d", n_chunks, oo_ctx::kMaxChunks);
    c->host_chunks = (int)n_chunks;
    return OO_OK;
}
extern "C" OO_API oo_status oo_set_host_zero_copy(oo_ctx* c, uint32_t enable) {
    if (!c) return OO_ERR_INVALID_ARG;
    c->host_zero_copy = enable != 0;
    return OO_OK;
}

extern "C" OO_API oo_status oo_query_host(oo_ctx* c, const oo_queries* q, float* h_rgb, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!q) return fail(c, OO_ERR_INVALID_ARG, "queries is NULL");
    if (q->perm) return fail(c, OO_ERR_INVALID_ARG, "oo_query_host: perm must be NULL");
    if (oo_status st = check_queries(c, q, true)) return st;
    if (q->n == 0) return OO_OK;
    if (!h_rgb) return fail(c, OO_ERR_INVALID_ARG, "rgb is NULL");
    if (!c->have_mlp) return fail(c, OO_ERR_NOT_READY, "no MLP uploaded");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g(c->device);
    // ---- zero-copy: when every buffer is PINNED host memory the kernels can address, ONE launch reads the queries straight from
    // host memory (the next tile's queries are prefetched behind the current tile, so the PCIe reads stream at the link rate) and
    // writes the RGB straight back: no staging copies, no chunks, no extra streams.  Measured on B200, config 1 (37.7 MB in,
    // 12.6 MB out): 0.80 ms against 0.93-1.17 ms for the chunked pipeline below and a copy-in floor of 0.69 ms.  Not used when the
    // batch is going to be binned (the bin pass would read the queries over PCIe twice) or any buffer is pageable.
    if (c->host_zero_copy) {
        auto dev_alias = [&](const void* h, const void** d) -> bool {
            if (!h) { *d = nullptr; return true; }
            cudaPointerAttributes a{};
            if (cudaPointerGetAttributes(&a, h) != cudaSuccess) { (void)cudaGetLastError(); return false; }
            if (a.type != cudaMemoryTypeHost || !a.devicePointer) return false;
            *d = a.devicePointer;
            return true;
        };
        const void *dx, *dn, *dw, *de, *dd, *dr;
        if (dev_alias(q->x, &dx) && dev_alias(q->nrm, &dn) && dev_alias(q->wo, &dw) && dev_alias(q->n_extra ? q->extra : nullptr, &de) &&
            dev_alias(q->disparity, &dd) && dev_alias(h_rgb, &dr) && !bin_wanted(c, q)) {
            oo_queries dq = *q;
            dq.x = (const float*)dx; dq.nrm = (const float*)dn; dq.wo = (const float*)dw; dq.extra = (const float*)de; dq.disparity = (const float*)dd;
            const oo_status st = query_device(c, &dq, (float*)const_cast<void*>(dr), stream);
            const cudaError_t e = cudaStreamSynchronize(stream);
            if (st) return st;
            OO_CUDA(c, e);
            c->info.host_zero_copy_last = 1;
            return OO_OK;
        }
    }
    c->info.host_zero_copy_last = 0;
    if (q->n > c->reserved) return fail(c, OO_ERR_NOT_READY, "the copy pipeline stages the batch in scratch: call oo_reserve(%llu) first", (unsigned long long)q->n);
    if (!c->have_pipe) {
        OO_CUDA(c, cudaStreamCreateWithFlags(&c->s_h2d, cudaStreamNonBlocking));
        OO_CUDA(c, cudaStreamCreateWithFlags(&c->s_d2h, cudaStreamNonBlocking));
        OO_CUDA(c, cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming));
        OO_CUDA(c, cudaEventCreateWithFlags(&c->ev_out, cudaEventDisableTiming));
        for (int i = 0; i < oo_ctx::kMaxChunks; ++i) {
            OO_CUDA(c, cudaEventCreateWithFlags(&c->ev_in[i], cudaEventDisableTiming));
            OO_CUDA(c, cudaEventCreateWithFlags(&c->ev_k[i], cudaEventDisableTiming));
        }
        c->have_pipe = true;
    }
    // Chunked three-stage pipeline: copy-in of chunk i+1 (s_h2d) overlaps the kernel of chunk i (caller's stream) and the
    // copy-out of chunk i-1 (s_d2h); PCIe is full duplex, so a frame costs about its copy-in time instead of the sum of the three.
    // Chunks are whole multiples of 128-query tiles, all of one size.  The chunk count follows the batch size (oo_set_host_chunks
    // overrides): one chunk below 128 Ki queries, else about 256 Ki queries per chunk, at least 2 and at most 8 chunks.
    // Measured on B200 (config 1 = 2^20 queries, pinned buffers): 1 chunk 1.07-1.10 ms, 2: 0.99, 4: 0.93-0.98, 8: 1.01-1.03, 16: 1.15 ms;
    // five chunks with a half-length first and last one (to shorten the exposed head and tail) 1.09 ms: every chunk costs three
    // host-to-device copies whose fixed cost outweighs what a shorter head saves.  The floor is the 37.7 MB copy-in at the
    // measured 54.8 GB/s = 0.69 ms.
    const uint64_t n = q->n;
    int want = c->host_chunks;
    if (want <= 0) want = n < (1u << 17) ? 1 : (int)std::min<uint64_t>(8, std::max<uint64_t>(2, n >> 18));
    uint64_t bounds[oo_ctx::kMaxChunks + 1];
    int n_chunks = 0;
    {
        uint64_t unit = (n + want - 1) / want;
        unit = (unit + 127) & ~127ull;
        bounds[0] = 0;
        for (int i = 0; i < want && bounds[n_chunks] < n; ++i) {
            bounds[n_chunks + 1] = std::min(n, bounds[n_chunks] + unit);
            ++n_chunks;
        }
        bounds[n_chunks] = n;
    }
    const uint32_t od = c->M.out_dim;
    // any failure below leaves copies from / to the caller's host buffers in flight on the library's streams: drain all three
    // before returning, so that the caller may free or reuse its buffers whatever the status
    auto drain = [&](oo_status st) {
        cudaStreamSynchronize(c->s_h2d); cudaStreamSynchronize(c->s_d2h); cudaStreamSynchronize(stream);
        return st;
    };
#define OO_PIPE(call)                                                                                                         \
    do {                                                                                                                      \
        cudaError_t e_ = (call);                                                                                              \
        if (e_ != cudaSuccess) {                                                                                              \
            (void)cudaGetLastError();                                                                                         \
            if (is_fatal(e_)) c->sticky = e_;                                                                                 \
            return drain(fail(c, OO_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)));                                      \
        }                                                                                                                     \
    } while (0)
    OO_PIPE(cudaEventRecord(c->ev_start, stream));
    OO_PIPE(cudaStreamWaitEvent(c->s_h2d, c->ev_start, 0));
    OO_PIPE(cudaStreamWaitEvent(c->s_d2h, c->ev_start, 0));
    for (int i = 0; i < n_chunks; ++i) {
        const uint64_t o = bounds[i], m = bounds[i + 1] - o;
        OO_PIPE(cudaMemcpyAsync(c->d_qx + o * 3, q->x + o * 3, m * 12, cudaMemcpyHostToDevice, c->s_h2d));
        OO_PIPE(cudaMemcpyAsync(c->d_qn + o * 3, q->nrm + o * 3, m * 12, cudaMemcpyHostToDevice, c->s_h2d));
        OO_PIPE(cudaMemcpyAsync(c->d_qw + o * 3, q->wo + o * 3, m * 12, cudaMemcpyHostToDevice, c->s_h2d));
        if (q->n_extra) OO_PIPE(cudaMemcpyAsync(c->d_qe + o * q->n_extra, q->extra + o * q->n_extra, m * 4 * q->n_extra, cudaMemcpyHostToDevice, c->s_h2d));
        if (q->disparity) OO_PIPE(cudaMemcpyAsync(c->d_qd + o, q->disparity + o, m * 4, cudaMemcpyHostToDevice, c->s_h2d));
        OO_PIPE(cudaEventRecord(c->ev_in[i], c->s_h2d));
        OO_PIPE(cudaStreamWaitEvent(stream, c->ev_in[i], 0));
        oo_queries dq = *q;
        dq.n = m;
        dq.x = c->d_qx + o * 3; dq.nrm = c->d_qn + o * 3; dq.wo = c->d_qw + o * 3;
        dq.extra = q->n_extra ? c->d_qe + o * q->n_extra : nullptr;
        dq.disparity = q->disparity ? c->d_qd + o : nullptr;
        if (oo_status st = query_device(c, &dq, c->d_rgb + o * od, stream)) return drain(st);
        OO_PIPE(cudaEventRecord(c->ev_k[i], stream));
        OO_PIPE(cudaStreamWaitEvent(c->s_d2h, c->ev_k[i], 0));
        OO_PIPE(cudaMemcpyAsync(h_rgb + o * od, c->d_rgb + o * od, m * 4 * od, cudaMemcpyDeviceToHost, c->s_d2h));
    }
    OO_PIPE(cudaEventRecord(c->ev_out, c->s_d2h));
    OO_PIPE(cudaStreamWaitEvent(stream, c->ev_out, 0));
    OO_PIPE(cudaStreamSynchronize(stream));
#undef OO_PIPE
    return OO_OK;
}

extern "C" OO_API oo_status oo_upload_scene(oo_ctx* c, const oo_scene_desc* sc, void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!sc) return fail(c, OO_ERR_INVALID_ARG, "scene is NULL");
    if (sc->n_spheres > 2048) return fail(c, OO_ERR_UNSUPPORTED, "%u spheres: at most 2048 (they are kept in shared memory)", sc->n_spheres);
    if (sc->n_spheres && !sc->spheres) return fail(c, OO_ERR_INVALID_ARG, "scene.spheres is NULL");
    if (!(sc->lo < sc->hi)) return fail(c, OO_ERR_INVALID_ARG, "scene box: need lo < hi");
    for (uint32_t s = 0; s < sc->n_spheres; ++s)
        if (!(sc->spheres[4 * s + 3] > 0.0)) return fail(c, OO_ERR_INVALID_ARG, "sphere %u: radius must be positive", s);
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    DeviceGuard g(c->device);
    free_dev(c->d_spheres);
    c->have_scene = false;
    OO_CUDA(c, cudaMalloc(&c->d_spheres, std::max<size_t>(sc->n_spheres, 1) * 4 * sizeof(double)));
    if (sc->n_spheres) OO_CUDA(c, cudaMemcpyAsync(c->d_spheres, sc->spheres, (size_t)sc->n_spheres * 4 * sizeof(double), cudaMemcpyHostToDevice, stream));
    OO_CUDA(c, cudaStreamSynchronize(stream));
    c->n_spheres = sc->n_spheres; c->scene_lo = sc->lo; c->scene_hi = sc->hi;
    c->have_scene = true;
    return OO_OK;
}

extern "C" OO_API oo_status oo_raycast(oo_ctx* c, const oo_camera_desc* cam, float* d_x, float* d_nrm, float* d_wo, int32_t* d_surf,
                                void* cuda_stream) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!c->have_scene) return fail(c, OO_ERR_NOT_READY, "no scene uploaded");
    if (!cam) return fail(c, OO_ERR_INVALID_ARG, "camera is NULL");
    const uint64_t n = (uint64_t)cam->width * cam->height;
    if (n >= (1ull << 32)) return fail(c, OO_ERR_UNSUPPORTED, "more than 2^32-1 pixels per frame");
    if (n && (!d_x || !d_nrm || !d_wo)) return fail(c, OO_ERR_INVALID_ARG, "output buffer is NULL");
    if (!(cam->vfov_deg > 0.0 && cam->vfov_deg < 180.0)) return fail(c, OO_ERR_INVALID_ARG, "vfov_deg must lie in (0, 180)");
    double fl = 0.0, cr = 0.0;
    {
        const double f[3] = {cam->look[0] - cam->eye[0], cam->look[1] - cam->eye[1], cam->look[2] - cam->eye[2]};
        fl = f[0] * f[0] + f[1] * f[1] + f[2] * f[2];
        const double r[3] = {f[1] * cam->up[2] - f[2] * cam->up[1], f[2] * cam->up[0] - f[0] * cam->up[2], f[0] * cam->up[1] - f[1] * cam->up[0]};
        cr = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
    }
    if (!(fl > 0.0) || !(cr > 0.0)) return fail(c, OO_ERR_INVALID_ARG, "degenerate camera: look == eye, or up parallel to the view direction");
    if (oo_status st = check_before(c)) return st;
    if (n == 0) return OO_OK;
    DeviceGuard g(c->device);
    const int k = launch_raycast((const double*)c->d_spheres, c->n_spheres, c->scene_lo, c->scene_hi, cam->eye, cam->look, cam->up,
                                 cam->vfov_deg, cam->width, cam->height, d_x, d_nrm, d_wo, d_surf, (cudaStream_t)cuda_stream);
    if (k < 0) return launch_failed(c, k, "ray-cast kernel (scene size)");
    count(c, k);
    return check_after(c);
}

extern "C" OO_API oo_status oo_read_padded_map(oo_ctx* c, uint32_t level, uint32_t slot, void* h_out) {
    if (!c) return OO_ERR_INVALID_ARG;
    if (!c->have_tree) return fail(c, OO_ERR_NOT_READY, "no tree uploaded");
    if (level >= c->T.n_levels || slot >= c->level_slots[level] || !h_out) return fail(c, OO_ERR_INVALID_ARG, "bad level/slot/pointer");
    if (c->T.vertex) return fail(c, OO_ERR_UNSUPPORTED, "vertex maps have no padded copy (they are stored unpadded, their seam tied at upload)");
    DeviceGuard g(c->device);
    const LevelParams& lv = c->T.lv[level];
    OO_CUDA(c, cudaMemcpy(h_out, (const uint8_t*)c->atlas_dev[level] + (uint64_t)(slot + 1) * lv.map_bytes, lv.map_bytes, cudaMemcpyDeviceToHost));   // + 1: the zero map
    return OO_OK;
}
