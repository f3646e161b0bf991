/*
 * oo.h — C ABI of liboo: batched per-query radiance evaluation of an OctaOctree neural radiosity cache on one
 * NVIDIA B200 (sm_100a).
 *
 * What the library computes (paper: /root/reference/PAPER.md, cited P:line; readings A1-A24 in DESIGN.md §2):
 * "rendering reduces to standard primary visibility plus one OctaOctree query and one decoder evaluation per visible
 * shading point".  For each query (position x, normal n, outgoing direction wo[, extras]):
 *   1. locate the cell containing x at every used octree level (sparse octree);
 *   2. project wo onto the unfolded octahedron (Eq. 4-5), remap to [0,1]^2, and interpolate that
 *      cell's directional feature map bilinearly with octahedral border wrap (texel reading of Eq. 6; continuity
 *      across faces);
 *   3. concatenate the per-level features (Eq. 11) with the per-query attributes (Eq. 12-13);
 *   4. decode with a small MLP (hidden width 64, ReLU, no biases) to RGB.
 * This is the nearest-cell / raw-direction variant that the paper itself names as ablations; see
 * DESIGN.md §1 for the differences from the full method.  The paper's full query is selected piece by piece with
 * oo_set_mode (8-neighbour trilinear blend, Eq. 10; mirror / disparity-shifted lookup direction, Eq. 8-9; the attribute
 * vector of Eq. 12) and oo_tree_desc.dirmap (vertex-stored maps with barycentric taps, Eq. 6); decoders of width 64 or
 * 128.  See "The paper's full query" below.
 *
 * Conventions
 *   - Every pointer is marked HOST or DEVICE.  DEVICE pointers must belong to the context's CUDA device.
 *   - Uploads copy (and re-lay-out) into library-owned device memory; the caller may free its buffers once the
 *     stream has completed.  A second upload replaces the first.
 *   - Query and output buffers are owned by the caller.  Kernels are enqueued on the caller's stream (a cudaStream_t
 *     passed as void*; NULL = the legacy default stream) and the call returns without synchronising, except where
 *     stated.  Hot calls never allocate: whatever scratch a call needs comes from oo_reserve (oo_sort_queries,
 *     oo_query_host, OO_PRESORT_BIN, OO_PATH_GENERIC / OO_PATH_UNFUSED, disparity prediction); a call that finds it
 *     missing returns OO_ERR_NOT_READY and launches nothing.
 *   - Every call returns oo_status; nothing throws.  oo_last_error() describes the last failure on that context.  A
 *     failed call leaves the context usable unless the CUDA context itself is lost (illegal address, launch failure,
 *     ...: every later call then fails at once with OO_ERR_CUDA).  A non-fatal CUDA error that some other code left
 *     pending on the calling thread is cleared by the next oo_ call that launches (it is not this library's to report).
 *   - One context per device; several contexts, on the same or on different devices, may live in one process.
 *   - A context is not thread-safe, and its hot calls share context-owned scratch (the binned copy of the queries, staging, feature
 *     rows, coherence samples): calls on ONE context must be ordered on one stream (or by events between streams).  Work that is to
 *     overlap on several streams takes one context per stream.
 *   - Not checked per query (result undefined, never a crash): non-finite inputs, wo = 0.  x outside [0,1]^3 is
 *     clamped componentwise (A16).
 *   - There is no CPU fallback: without a usable CUDA device oo_create fails.
 */
#ifndef OO_H_
#define OO_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define OO_API __attribute__((visibility("default")))
#else
#define OO_API
#endif

#define OO_MAX_LEVELS 8      /* used levels L */
#define OO_MAX_DEPTH 16      /* octree depth (root = depth 0) */
#define OO_MAX_HIDDEN 8      /* hidden layers H */
#define OO_MAX_EXTRA 10      /* per-query extra scalars appended to the MLP input */

typedef struct oo_ctx oo_ctx; /* opaque; one per device */

typedef enum {
    OO_OK = 0,
    OO_ERR_INVALID_ARG = 1, /* null pointer, inconsistent sizes, malformed tree ... (see oo_last_error) */
    OO_ERR_NOT_READY = 2,   /* tree / MLP not uploaded yet, or MLP input width does not match the tree */
    OO_ERR_UNSUPPORTED = 3, /* valid request outside what the kernels implement (e.g. width != 64) */
    OO_ERR_CUDA = 4,        /* a CUDA call failed (also reports an earlier asynchronous fault) */
    OO_ERR_OOM = 5          /* host or device allocation failed */
} oo_status;

typedef enum { OO_F16 = 0, OO_F32 = 1 } oo_dtype;
typedef enum { OO_ACT_NONE = 0, OO_ACT_EXP = 1 } oo_out_act;

/* ---- The paper's full query.  All-zero = the hot path described above. ---- */
/* f1, Eq. 10: features sit at cell centres; with p = clamp(x,0,1)*2^d - 1/2, k0 = floor(p), t = p - k0 the
 * eight cells k0 + {0,1}^3 are blended with trilinear weights prod(t or 1-t), restricted to the non-empty cells inside
 * the grid and renormalised by the sum of the surviving weights (none survives => zero features). */
typedef enum { OO_SPATIAL_NEAREST = 0, OO_SPATIAL_TRILINEAR8 = 1 } oo_spatial;
/* f2, Eq. 6: OO_DIRMAP_VERTEX stores every map as (R+1) x (R+1) VERTICES of the unfolded octahedral
 * grid with R intervals per axis; the lookup finds the grid cell (ci, cj) = min(floor((u+1)/2*R), R-1), splits it along
 * the anti-diagonal where u_x*u_y > 0 (cell in a same-sign quadrant) and along the main diagonal otherwise, so that the
 * hypotenuses run parallel to the octahedron's face edges, and takes the barycentric combination of the containing
 * triangle's three vertices.  Boundary vertices that coincide on the sphere ("the edge vertices are shared along adjacent
 * faces", Fig. 3 caption / P:125) are stored separately in the caller's arrays: (0, c) and (0, R-c), (R, c) and (R, R-c),
 * (r, 0) and (R-r, 0), (r, R) and (R-r, R) are one vertex each, the four corners are all the -z pole.  oo_upload_tree TIES
 * them in the library's copy: each pair takes the value of the member with the smaller index along its side, the corners
 * that of vertex (0, 0), so the interpolant is continuous across the seam whatever was stored (a cache whose owner shares
 * them already is unchanged).  oo_info.tied_vertices counts the stored vertices the last upload rewrote. */
typedef enum { OO_DIRMAP_TEXEL = 0, OO_DIRMAP_VERTEX = 1 } oo_dirmap;
/* f3, P:135 and Eq. 8-9: the direction that indexes the maps.  WO: wo itself.  MIRROR: w_r = 2(n.wo)n - wo.
 * SHIFTED: per cell j with centre c_j, w~_j = (x - c_j)*d^ + w_r (Eq. 9 before normalisation; Eq. 4 is scale invariant),
 * d^ = oo_queries.disparity (the output of the disparity predictor of Eq. 7, supplied per query).  Directions are formed
 * in fp32, one rounding per operation, in the order DESIGN.md "Index contract (full query)" fixes. */
typedef enum { OO_LOOKUP_WO = 0, OO_LOOKUP_MIRROR = 1, OO_LOOKUP_SHIFTED = 2 } oo_lookup;
/* f4, Eq. 12: decoder input after the features.  N_WO: [n | wo | extra].  PAPER: [x | w_r | n | extra]
 * (extra = albedo a, roughness alpha, ... as supplied). */
typedef enum { OO_ATTRS_N_WO = 0, OO_ATTRS_PAPER = 1 } oo_attrs;
typedef struct {
    oo_spatial spatial;
    oo_lookup lookup;
    oo_attrs attrs;
} oo_mode;

/* Which kernels oo_encode / oo_query run.  Every choice computes the same function; all are CUDA. */
typedef enum {
    OO_PATH_AUTO = 0,        /* fastest available for the uploaded shapes */
    OO_PATH_GENERIC = 1,     /* any tree: plain child-table descent; encode -> features in HBM -> MLP kernel */
    OO_PATH_UNFUSED = 2,     /* hop-table descent, specialised gather; features round-trip HBM; MLP kernel */
    OO_PATH_FUSED_MMA = 3,   /* one kernel: gather -> shared memory -> mma.sync MLP -> RGB */
    OO_PATH_FUSED_TC = 4,    /* one kernel: gather -> shared memory -> tcgen05.mma (TMEM accumulators) -> RGB */
    OO_PATH_FUSED_TC_TMEM = 5, /* the same with the activations (A operand) kept in tensor memory: no shared-memory A tile */
    OO_PATH_FULL = 6         /* reported by oo_get_info when the full-query kernels ran (mode != 0, vertex maps or width 128);
                                not selectable with oo_set_path */
} oo_path;

/* Row a1 inside oo_query (BASELINE.json north_star: "an optional Morton pre-sort of queries for gather locality").
 * OO_PRESORT_NONE: queries are processed in the caller's order (or in queries.perm's).
 * OO_PRESORT_BIN: oo_query first bins the queries by the top 10 bits of their 30-bit Morton key (the octree cell at depth 3
 *   plus one bit: ONE counting pass, 3 launches) MOVING x, n, wo and the extras into library scratch, runs the chosen
 *   kernel path over the binned copy, and a last kernel brings the RGB back to the caller's order.  Results are
 *   bit-identical to OO_PRESORT_NONE (queries are independent); what changes is which atlas pages the thread blocks touch
 *   at a time.  For incoherent queries out of an HBM-resident cache (configs[4]); screen-order frames are coherent already.
 *   Takes effect (hot path and full query alike; a supplied queries.disparity moves with its query, a predicted one is
 *   predicted on the binned copy) when queries.perm is NULL and n >= min_queries of oo_set_presort (default 262144:
 *   below that the extra launches cost more than they save); otherwise the call proceeds in the given order (oo_info.presorted_last_query says
 *   which).  oo_encode on OO_PATH_UNFUSED does the same with x and wo and stores every feature row at its query's index
 *   (oo_info.presorted_last_encode).  Needs oo_reserve(n).
 * OO_PRESORT_AUTO (default): the library decides per call between the two from the coherence of the recent calls' queries.
 *   Every kernel that reads the queries in the caller's order samples, in a few of its warps, how many distinct depth-4
 *   octree cells 32 consecutive queries fall into (1-3 for screen-order primary hits, ~30 for random surface samples) and
 *   leaves the sample in a small device array that a library-owned side stream copies to the host after the call's kernels;
 *   the next call reads what has arrived -- nothing waits, the call stays asynchronous, the caller's stream carries one extra
 *   event record -- and bins when the mean exceeds 12 (and stops below 6).  The decision therefore lags one call: the first
 *   incoherent batch of a stream runs unsorted.  Without reserved scratch AUTO proceeds unsorted instead of failing.  The
 *   result bytes never depend on the decision.  oo_info.presort_auto_on / coherence_x100 report it.  Sampled by: the fused
 *   tensor-memory kernel, the histogram pass of a binned call, oo_encode's specialised kernel, the full-query kernel.
 *   CUDA graphs: a call made while its stream is being captured enqueues its kernels only (no event, no side-stream copy),
 *   so the capture ends cleanly; the captured graph contains the decision that was current at capture time and replays
 *   never change it.  Make one ordinary call of the same shape before capturing (first launches configure the kernels). */
typedef enum { OO_PRESORT_NONE = 0, OO_PRESORT_BIN = 1, OO_PRESORT_AUTO = 2 } oo_presort;

/* The octree and its feature atlases ("every non-empty cell stores a learnable octahedral feature map").
 * Node 0 is the root (depth 0, the cube [0,1]^3); a node of depth d is a cell of side 2^-d with half-open extent.
 * Octant index o = bx | by<<1 | bz<<2 (b = 1 for the upper half along that axis).  Used levels are listed coarse to
 * fine; every existing node at a used depth owns one map: atlas[l][map_slot[node]] is an R_l x R_l array of F-vectors,
 * row j (v_y) major, column i (v_x) minor, texel centres at ((i+1/2)/R, (j+1/2)/R) of the unfolded octahedron (A2, A3). */
typedef struct {
    uint32_t n_nodes;
    uint32_t max_depth;          /* <= OO_MAX_DEPTH */
    const int32_t* child;        /* HOST [n_nodes][8]; -1 = absent; a child is one level deeper than its parent */
    const uint8_t* depth;        /* HOST [n_nodes] */
    const int32_t* map_slot;     /* HOST [n_nodes]; slot in its level's atlas; -1 where depth is not a used level */
    uint32_t n_levels;           /* L in 1..OO_MAX_LEVELS */
    const uint32_t* level_depth; /* HOST [L] strictly increasing, 1 <= depth <= max_depth */
    const uint32_t* level_res;   /* HOST [L] R_l: power of two, 2 <= R_l <= 256 */
    const uint32_t* level_slots; /* HOST [L] number of maps in level l (= number of nodes at that depth) */
    uint32_t n_features;         /* F; F * sizeof(dtype) must be 16, 32 or 64 bytes */
    oo_dtype dtype;              /* storage type of the texels */
    const void* const* atlas;    /* HOST array [L] of DEVICE pointers, each [level_slots[l]][R_l][R_l][F], 16-byte aligned
                                    (OO_DIRMAP_VERTEX: [level_slots[l]][R_l+1][R_l+1][F]) */
    oo_dirmap dirmap;            /* OO_DIRMAP_TEXEL (0): texel-centred maps, bilinear taps, border wrap; OO_DIRMAP_VERTEX */
} oo_tree_desc;

/* Decoder f_phi: n_hidden x (linear width x in, ReLU), then linear out_dim x width, then out_act.
 * No biases (A10).  fp16 weights, row-major [out][in].  in_dim must equal L*F + 6 + n_extra of the queries:
 * input order [h_0 .. h_{L-1} | n | wo | extra] (A7); with OO_ATTRS_PAPER L*F + 9 + n_extra: [h | x | w_r | n | extra]. */
typedef struct {
    uint32_t in_dim;
    uint32_t width;              /* 64, or 128 (the paper's decoder; runs on the full-query kernels) */
    uint32_t n_hidden;           /* 1..OO_MAX_HIDDEN */
    uint32_t out_dim;            /* 1..8 (3 = RGB); the full-query kernels: 1..4 */
    const void* const* weights;  /* HOST array [n_hidden+1] of pointers to fp16 matrices:
                                    [width][in_dim], (n_hidden-1) x [width][width], [out_dim][width] */
    oo_out_act out_act;
    uint32_t weights_on_device;  /* 0: weights[k] are HOST pointers; 1: DEVICE pointers on the context's device (e.g. a
                                    trainer's parameters), read on the upload stream */
} oo_mlp_desc;

/* A batch of queries.  All arrays packed fp32.  For oo_encode / oo_query / oo_sort_queries they are DEVICE pointers,
 * for oo_query_host HOST pointers.  Read-only for the library. */
typedef struct {
    uint64_t n;
    const float* x;              /* [n][3] position */
    const float* nrm;            /* [n][3] surface normal (may be NULL for oo_encode) */
    const float* wo;             /* [n][3] outgoing direction, need not be normalised (A22), must not be 0 */
    const float* extra;          /* [n][n_extra] or NULL */
    uint32_t n_extra;            /* 0..OO_MAX_EXTRA (roughness: 1) */
    const uint32_t* perm;        /* optional DEVICE [n]: processing order (thread t handles query perm[t]); results are
                                    always written at the query's own index, i.e. in the caller's order.  NULL = identity */
    const float* disparity;      /* [n] d^ of Eq. 7-9, required by OO_LOOKUP_SHIFTED, ignored otherwise (may be NULL) */
} oo_queries;

/* ---- Primary visibility of an analytic scene ("standard primary visibility"). ----
 * The scene BASELINE.json's configs describe: spheres plus a 5-plane box (x=lo, x=hi, y=lo, y=hi, z=lo, each a rectangle
 * spanning [lo,hi] on the other two axes, open towards +z).  The paper traces its G-buffers with Mitsuba 3;
 * this is the stand-in that lets a frame be produced on the device. */
typedef struct {
    uint32_t n_spheres;          /* 0..2048 */
    const double* spheres;       /* HOST [n_spheres][4] = centre x, y, z, radius */
    double lo, hi;               /* the box planes */
} oo_scene_desc;

/* Pinhole camera: f = normalize(look - eye), r = normalize(f x up), u = r x f; pixel (i, j) of a width x height frame is
 * sampled at its centre, d = normalize(f + px r + py u) with px = (2(i+1/2)/width - 1) tan(vfov/2) width/height and
 * py = (1 - 2(j+1/2)/height) tan(vfov/2); scanline order (query index = j*width + i). */
typedef struct {
    double eye[3], look[3], up[3];
    double vfov_deg;             /* vertical field of view, degrees */
    uint32_t width, height;
} oo_camera_desc;

typedef struct {
    uint64_t launches;           /* kernels launched by this context so far (all kinds) */
    uint64_t query_launches;     /* kernels launched by oo_query / oo_encode / oo_sort_queries / oo_query_host */
    uint64_t node_table_bytes;   /* device bytes of the descent tables */
    uint64_t atlas_bytes;        /* device bytes of the re-laid-out (border-padded) atlases */
    uint32_t path_last_query;    /* oo_path actually used by the last oo_query */
    uint32_t path_last_encode;   /* oo_path actually used by the last oo_encode */
    uint32_t hop_plan_ok;        /* 1 if the uploaded tree admits the hop-table descent (else only OO_PATH_GENERIC) */
    uint32_t n_sms;
    uint32_t presorted_last_query; /* 1 if the last oo_query ran on binned queries (OO_PRESORT_BIN took effect) */
    uint32_t presorted_last_encode; /* the same for the last oo_encode */
    uint32_t full_query;         /* 1 if oo_query runs the full-query kernel under the current tree / mode / decoder
                                    (mode != 0, vertex maps or width 128), i.e. oo_query_debug's outputs are [n][L][J]... */
    uint32_t n_neighbours;       /* J of the current mode: 8 (OO_SPATIAL_TRILINEAR8) or 1 */
    uint64_t tied_vertices;      /* OO_DIRMAP_VERTEX: boundary vertices the last oo_upload_tree rewrote when it tied the seam (0 for
                                    a cache stored with shared edge vertices, and for texel maps) */
    uint32_t host_zero_copy_last; /* 1 if the last oo_query_host read its (pinned) host buffers in place, 0 if it ran the copy pipeline */
    uint32_t presort_auto_on;    /* OO_PRESORT_AUTO's current decision: 1 = the next batch of >= min_queries queries is binned */
    uint32_t coherence_x100;     /* 100 x mean number of distinct depth-4 cells per 32 consecutive queries, latest sample */
    uint32_t encode_pipelined_last; /* 1 if the last oo_encode ran the pipelined-descent kernel (the batch was binned, or the latest coherence
                                    sample says its taps miss the caches), 0 if it ran the occupancy kernel (coherent frames); same bytes either way */
} oo_info;

/* Create a context on a CUDA device.  Fails with OO_ERR_CUDA if the device is absent or is not compute capability
 * 10.x (the kernels are built for sm_100a only). */
OO_API oo_status oo_create(oo_ctx** out, int cuda_device);
OO_API void oo_destroy(oo_ctx* ctx);
/* Message for the last non-OK status on ctx (valid until the next call on ctx); "" if none. */
OO_API const char* oo_last_error(const oo_ctx* ctx);
/* Informational, never an error: when the last oo_query resolved OO_PATH_AUTO to anything slower than the fused
 * tensor-memory kernel (a shape without such an instance, a tree without a hop plan, ...) this says to what and for which
 * shape; "" otherwise.  Valid until the next call on ctx. */
OO_API const char* oo_last_note(const oo_ctx* ctx);

/* Validate the tree (child indices in range and one level deeper, depth consistent, map_slot unique per level and
 * < level_slots), build the descent tables, and copy every atlas into library-owned border-padded maps
 * ((R+2)^2 texels per map, the one-texel border filled by the octahedral wrap).  Synchronises the stream. */
OO_API oo_status oo_upload_tree(oo_ctx* ctx, const oo_tree_desc* tree, void* cuda_stream);
/* Copy the decoder weights into the library's padded shared-memory image.  Synchronises the stream. */
OO_API oo_status oo_upload_mlp(oo_ctx* ctx, const oo_mlp_desc* mlp, void* cuda_stream);
/* Pre-allocate every scratch buffer a hot call may need for up to max_queries queries: sort keys, staging for
 * oo_query_host, the binned copy of OO_PRESORT_BIN (about 250 bytes per query in all), and, sized from the uploaded tree,
 * the feature rows of OO_PATH_GENERIC / OO_PATH_UNFUSED (L * texel bytes per query): call it after oo_upload_tree, and
 * again after uploading a tree with wider feature rows.  Never shrinks.  OO_ERR_OOM leaves the context usable. */
OO_API oo_status oo_reserve(oo_ctx* ctx, uint64_t max_queries);
/* Select the kernels used from now on (default OO_PATH_AUTO).  OO_ERR_UNSUPPORTED at query time if the uploaded
 * shapes have no such kernel. */
OO_API oo_status oo_set_path(oo_ctx* ctx, oo_path path);
OO_API oo_status oo_get_info(const oo_ctx* ctx, oo_info* out);

/* Select the in-query pre-sort policy (default OO_PRESORT_AUTO); see oo_presort.  Batches of fewer than min_queries queries proceed unsorted;
 * 0 selects the library default (262144, about where binning starts to pay on a B200).  OO_ERR_INVALID_ARG for an unknown
 * presort value. */
OO_API oo_status oo_set_presort(oo_ctx* ctx, oo_presort presort, uint64_t min_queries);
/* Select the variant of the query (default all-zero = the hot path).  Takes effect from the next oo_encode_full /
 * oo_query.  OO_LOOKUP_SHIFTED needs oo_queries.disparity; OO_ATTRS_PAPER changes the expected MLP in_dim. */
OO_API oo_status oo_set_mode(oo_ctx* ctx, const oo_mode* mode);

/* Row a1: d_perm_out[k] = index of the k-th query in ascending order of the 30-bit Morton key of
 * clamp(floor(x*1024), 0, 1023) (bit b of q_x -> key bit 3b, q_y -> 3b+1, q_z -> 3b+2), ties in original order
 * (stable).  d_perm_out: DEVICE [n].  Needs oo_reserve(n). */
OO_API oo_status oo_sort_queries(oo_ctx* ctx, const oo_queries* q, uint32_t* d_perm_out, void* cuda_stream);

/* Row a1 for callers that cannot allocate device memory.  Same result as oo_sort_queries (same kernels, same unique stable
 * permutation), but it needs no context, no oo_reserve and no cudaMalloc, cudaFree or allocating library routine, on any call:
 * its scratch is an array built into the library image.  It is meant for code that runs after an application has frozen its
 * memory budget, inside a host program that owns the device heap, or on a latency-critical thread where an allocation's
 * device-wide synchronisation is not acceptable.
 *   d_x         DEVICE [n][3] packed fp32 positions, read-only; d_perm_out DEVICE [n] uint32.  Both belong to the calling
 *               thread's CURRENT CUDA device, which is the device the call runs on.
 *   n           at most OO_SORT_STATIC_MAX_QUERIES; more returns OO_ERR_UNSUPPORTED and launches nothing (use oo_sort_queries).
 *   cuda_stream a cudaStream_t of that device (NULL = legacy default stream); kernels are enqueued, the call does not wait.
 *   err_msg     optional HOST buffer of err_cap bytes that receives a NUL-terminated description when the status is not
 *               OO_OK (emptied on success); NULL / 0 = status code only.
 * Cost: each GPU on which the call is made holds the scratch, 13,643,776 bytes, from its first call until the process exits.
 * First call on a device: it looks up the array's device address (cudaGetSymbolAddress) before it launches, which also makes
 * the CUDA runtime load that part of the library onto the device.  Make that first call (n = 0 is enough, and launches nothing)
 * during start-up, before any stream capture begins on that device; later calls only clear 12 KB and launch 9 kernels.
 * All calls a process makes on one device share the one array, and it keeps the previous call's contents (the call clears the
 * part that must start at zero itself).  Two such calls whose kernels can overlap on the GPU - issued to different streams
 * with no event between them, for instance from two host threads - race on the array and both permutations are garbage:
 * order the calls on one stream or with events.  (Another process has its own copy of the array.) */
#define OO_SORT_STATIC_MAX_QUERIES 1048576u   /* one 1024 x 1024 frame */
OO_API oo_status oo_sort_queries_static(const float* d_x, uint64_t n, uint32_t* d_perm_out, void* cuda_stream, char* err_msg,
                                        size_t err_cap);

/* Steps 1-3 only.  d_features: DEVICE [n][L*F] in the tree's dtype (fp32 accumulate, one rounding on store).
 * Optional debug outputs: d_slot DEVICE [n][L] (atlas slot per level, -1 = no cell at that level, whose features are
 * then 0, A17); d_texel DEVICE [n][L][2] = base texel (i0, j0) before wrapping, each in [-1, R_l-1], decided in fp32 by
 * the fixed sequence of DESIGN.md "Index contract".  q->nrm and q->extra are ignored. */
OO_API oo_status oo_encode(oo_ctx* ctx, const oo_queries* q, void* d_features, int32_t* d_slot, int16_t* d_texel,
                    void* cuda_stream);

/* Steps 1-3 under the current oo_mode and the tree's dirmap (any combination, the all-zero mode included).
 * d_features: DEVICE [n][L*F] fp32.  J = 8 neighbours (OO_SPATIAL_TRILINEAR8, j = a | b<<1 | c<<2 for cell k0 + (a,b,c))
 * or 1 (nearest).  Optional debug outputs: d_slot DEVICE [n][L][J] atlas slot of each neighbour (-1 = outside the grid or
 * empty); d_cell DEVICE [n][L][J][3] = the directional index decision for that neighbour's lookup direction: texel maps
 * (i0, j0, 0) as in oo_encode, vertex maps (ci, cj, upper) with upper = 1 for the triangle that holds local corner (1,1)
 * [anti-diagonal split] / (0,1) [main-diagonal split]. */
OO_API oo_status oo_encode_full(oo_ctx* ctx, const oo_queries* q, float* d_features, int32_t* d_slot, int16_t* d_cell,
                         void* cuda_stream);

/* The whole path.  d_rgb: DEVICE [n][out_dim] fp32, written at each query's own index.  Runs the hot-path kernels when
 * the mode is all-zero, the maps are texel maps and the decoder is 64 wide; otherwise the full-query kernel (one fused
 * launch as well). */
OO_API oo_status oo_query(oo_ctx* ctx, const oo_queries* q, float* d_rgb, void* cuda_stream);

/* oo_query that also reports which cell and which texels every query read -- from inside the very kernels oo_query
 * runs: every fused kernel has a second, compile-time instance whose gather code hands the atlas slot and the base texel
 * to an index sink at the point where it forms the texel address; this call selects those instances (same descent, same
 * address arithmetic, same RGB bit for bit; slower by the extra stores).  It exists so that BASELINE.json's "node indices
 * and texel indices bit-exact" can be checked on the timed kernels themselves rather than on oo_encode's.
 * Hot path: d_slot DEVICE [n][L], d_index DEVICE [n][L][2] = (i0, j0), as oo_encode.  Full query (mode != 0, vertex maps or
 * width 128): d_slot [n][L][J], d_index [n][L][J][3], as oo_encode_full.  Either may be NULL.  Rows land at the query's
 * own index whatever the processing order (perm, OO_PRESORT_BIN). */
OO_API oo_status oo_query_debug(oo_ctx* ctx, const oo_queries* q, float* d_rgb, int32_t* d_slot, int16_t* d_index,
                         void* cuda_stream);

/* Number of (equal) chunks oo_query_host splits a batch into: 1..16, or 0 (default) = chosen from the batch size (one
 * chunk below 131,072 queries, else about 262,144 queries per chunk, 2..8 chunks). */
OO_API oo_status oo_set_host_chunks(oo_ctx* ctx, uint32_t n_chunks);

/* oo_query_host reads PINNED host buffers in place (see there) when enable != 0 (default); 0 forces the chunked copy pipeline. */
OO_API oo_status oo_set_host_zero_copy(oo_ctx* ctx, uint32_t enable);

/* The whole path from HOST buffers.  Fast path (default, oo_set_host_zero_copy): when q->x, q->nrm, q->wo, q->extra,
 * q->disparity and h_rgb are all pinned (page-locked) host memory that the device can address, and the batch is not going to
 * be binned (oo_presort), ONE launch of the fused kernel reads the queries straight from host memory over PCIe -- the next
 * tile's queries are prefetched behind the current tile, so the reads stream -- and writes the RGB straight back: no staging
 * copy, no chunks (oo_info.host_zero_copy_last = 1).  Needs no oo_reserve.  Otherwise (pageable memory, binned batches, or the
 * fast path switched off) a chunked three-stage pipeline: the queries are split into chunks of whole
 * 128-query tiles (see oo_set_host_chunks); chunk i+1 is copied to the device on a library-owned copy-in
 * stream while oo_query runs chunk i on the caller's stream and chunk i-1's RGB returns to h_rgb (HOST [n][out_dim]) on
 * a library-owned copy-out stream.  Work starts after everything already enqueued on the caller's stream; the call
 * returns after all three streams have finished (it synchronises), on failure too: no copy from or to the caller's
 * buffers is in flight when it returns, whatever the status.  q->perm must be NULL.  Pinned host memory lets the
 * copies overlap; pageable memory works but serialises.  Needs oo_reserve(n).  Launches one fused kernel per chunk. */
OO_API oo_status oo_query_host(oo_ctx* ctx, const oo_queries* q, float* h_rgb, void* cuda_stream);

/* ---- The disparity predictor g_psi of Eq. 7 (the rest of SURVEY.md §8(f) row f3) ----
 * d^(x, w_r) = g_psi(x, w_r): "a compact multi-resolution hash-grid network in the style of Instant-NGP" with "2 hidden
 * layers of 64 neurons".  The paper gives no further hyper-parameter; the readings:
 *   - G levels over position; level g has res[g] = N_g intervals per axis, i.e. (N_g+1)^3 grid vertices over [0,1]^3, and
 *     a table of T_g entries of two fp16 features; T_g = (N_g+1)^3 when that is <= 2^hash_log2 (dense: vertex (i,j,k) owns
 *     entry i + (N_g+1)(j + (N_g+1)k)), else T_g = 2^hash_log2 and vertex (i,j,k) reads entry
 *     (i ^ j*2654435761 ^ k*805459861) mod 2^hash_log2, products modulo 2^32 (collisions are not resolved);
 *   - x is clamped to [0,1]^3; p = x*N_g in fp32, cell c0 = min(floor(p), N_g-1), t = p - c0; the level's feature is the
 *     trilinear interpolation of the cell's eight vertices;
 *   - network input [e_0 .. e_{G-1} | w_r] (2G + 3 scalars, w_r = 2(n.wo)n - wo raw), hidden layers 64 wide, ReLU, no
 *     biases, one output z, d^ = exp(z). */
#define OO_MAX_GRID_LEVELS 16
typedef struct {
    uint32_t n_levels;           /* G in 1..OO_MAX_GRID_LEVELS */
    uint32_t n_features;         /* features per entry: 2 */
    const uint32_t* res;         /* HOST [G]: N_g, coarse to fine, each in 1..2^20 */
    uint32_t hash_log2;          /* 4..28 */
    const void* const* tables;   /* HOST [G] of HOST fp16 [T_g][2] */
    uint32_t n_hidden;           /* 1..OO_MAX_HIDDEN (the paper: 2) */
    const void* const* weights;  /* HOST [n_hidden+1] of HOST fp16 matrices: [64][2G+3], (n_hidden-1) x [64][64], [1][64] */
} oo_disparity_desc;
/* Copy the tables and weights into library-owned device memory.  Synchronises the stream.  From then on oo_query /
 * oo_encode_full / oo_query_host with OO_LOOKUP_SHIFTED and queries.disparity == NULL predict d^ themselves (one extra
 * launch into scratch: needs oo_reserve(n)). */
OO_API oo_status oo_upload_disparity(oo_ctx* ctx, const oo_disparity_desc* d, void* cuda_stream);
/* d_disparity: DEVICE [n] fp32 = d^ per query (q->x, q->nrm, q->wo; perm and extras ignored).  d_features: optional
 * DEVICE [n][2G] fp32, the hash-grid features e(x) before they are rounded to fp16 for the network (NULL to skip). */
OO_API oo_status oo_predict_disparity(oo_ctx* ctx, const oo_queries* q, float* d_disparity, float* d_features, void* cuda_stream);

/* Copy the scene into library-owned device memory.  Synchronises the stream. */
OO_API oo_status oo_upload_scene(oo_ctx* ctx, const oo_scene_desc* scene, void* cuda_stream);
/* Trace one primary ray per pixel against the uploaded scene and write the queries of the frame: d_x (hit point), d_nrm
 * (sphere: outward normal (x - c)/R; plane: the unit axis vector pointing into the box), d_wo = -d, each DEVICE
 * [width*height][3] fp32, and optionally d_surf DEVICE [width*height] (sphere index, n_spheres + plane index, -1 = miss;
 * a miss writes zeros).  The nearest hit with t > 1e-9 wins; among equal t the earlier surface (spheres in order, then
 * the planes).  Arithmetic: double precision, every operation rounded on its own, outputs rounded once to fp32
 * (DESIGN.md "Ray cast").  The buffers can be passed to oo_query / oo_encode as they are. */
OO_API oo_status oo_raycast(oo_ctx* ctx, const oo_camera_desc* cam, float* d_x, float* d_nrm, float* d_wo, int32_t* d_surf,
                     void* cuda_stream);

/* Debug read-back of the library's re-laid-out atlas: copies the padded map of (level, slot) to HOST
 * h_out [(R+2)][(R+2)][F] in the tree's dtype.  Synchronous. */
OO_API oo_status oo_read_padded_map(oo_ctx* ctx, uint32_t level, uint32_t slot, void* h_out);

#ifdef __cplusplus
}
#endif
#endif /* OO_H_ */
