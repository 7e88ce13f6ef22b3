// tpc_cf_api.cu — the C ABI of include/tpc_cf.h: argument validation, workspace carving, kernel sequencing.
// The library never allocates device memory; the handle owns host state and a few CUDA events only.
#include <new>
#include <stdio.h>
#include <string.h>

#include <nvtx3/nvToolsExt.h>

#include "tpc_cf_internal.cuh"

using namespace tpccf;

// NVTX range over a group of launches (host side: marks the enqueue; a profiler correlates the kernels under it).
// A no-op unless a tool is attached.
struct NvtxRange {
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

static constexpr int kProfSlots = 64;
static constexpr int kMaxGroups = 18;    // sector groups of the tpc_cf_run_host pipeline

struct tpc_cf {
    Geo geo;
    Workspace ws;
    uint64_t max_digits, max_clusters;
    uint32_t n_sort_tiles;
    size_t map_bytes;
    int last_launches;
    uint64_t shape_n;           // digits of the whole frame while tpc_cf_run_host runs it group by group, else 0
    Tuning tun;                 // tpc_cf_debug_set overrides (all 0 by default)
    uint32_t ws_flags;          // TPC_CF_WS_* the workspace was carved with
    uint64_t shape_hint;        // tpc_cf_set_frame_digits: digits of the whole frame when runs cover a part of it, else 0
    const char* last_kernel;
    int profiling;
    uint32_t run_index;         // runs since profiling was switched on
    cudaEvent_t ev[kProfSlots][4];   // per slot: run begin, dominant kernel begin, dominant kernel end, run end
    // tpc_cf_run_host pipeline (created on first use): copy-in / copy-out streams, per-group events, pinned status
    bool pipe_ready;
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_fork, ev_join, ev_in[kMaxGroups], ev_run[kMaxGroups];
    tpc_cf_status* pinned_status;    // [kMaxGroups], cudaHostAlloc
    char cuda_msg[256];
};

static thread_local char g_last_cuda_msg[256] = "";

static bool geometry_to_geo(const tpc_cf_geometry* g, Geo* out)
{
    if (g->n_sectors == 0 || g->n_rows == 0 || g->max_pads == 0 || g->n_time == 0) return false;
    if (g->n_sectors > 256 || g->n_rows > 256 || g->max_pads > 255 || g->n_time > 65535) return false;
    memset(out, 0, sizeof *out);
    out->n_sectors = g->n_sectors; out->n_rows = g->n_rows; out->max_pads = g->max_pads; out->n_time = g->n_time;
    out->n_planes = g->n_sectors * g->n_rows;
    out->PS = g->max_pads + 4;
    out->TS = (g->n_time + 4 + 7) & ~7u;
    out->LS = g->max_pads + 1;
    for (uint32_t r = 0; r < g->n_rows; ++r) {
        const uint32_t p = g->npads ? g->npads[r] : g->max_pads;
        if (p == 0 || p > g->max_pads) return false;
        out->npads[r] = (uint8_t)p;
    }
    return true;
}

static bool same_geometry(const Geo& a, const Geo& b)
{
    return a.n_sectors == b.n_sectors && a.n_rows == b.n_rows && a.max_pads == b.max_pads &&
           a.n_time == b.n_time && memcmp(a.npads, b.npads, sizeof a.npads) == 0;
}

static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

// Carves the workspace; base may be NULL to compute the size only.
static size_t carve(const Geo& g, uint64_t max_digits, uint64_t max_clusters, uint32_t ws_flags, char* base,
                    Workspace* ws, uint32_t* n_sort_tiles, size_t* map_bytes)
{
    const bool sorted_only = (ws_flags & TPC_CF_WS_SORTED_ONLY) != 0;   // no map, no mask, no sort scratch
    size_t off = 0;
    auto take = [&](size_t bytes) { char* p = base ? base + off : nullptr; off += align256(bytes ? bytes : 1); return p; };
    const uint64_t nwords = ceil_div_u64(max_digits, 32) + 1;
    const uint64_t nblk = ceil_div_u64(nwords, 256) + 1;
    const uint64_t tiles = ceil_div_u64(max_clusters ? max_clusters : 1, 2048);
    const size_t mapb = sorted_only ? 0 : (size_t)g.n_planes * g.PS * g.TS * sizeof(uint16_t);
    if (sorted_only) max_clusters = 0;
    Workspace w;
    w.counters = (Counters*)take(sizeof(Counters));
    w.map = (uint16_t*)take(mapb);
    w.peakmask = (uint32_t*)take(sorted_only ? 0 : nwords * 4);
    w.blk_cnt = (uint32_t*)take(sorted_only ? 0 : nblk * 4);
    w.blk_off = (uint32_t*)take(sorted_only ? 0 : nblk * 4);
    w.scan_part = (uint32_t*)take(sorted_only ? 0 : (ceil_div_u64(nblk, 1024) + 1) * 4);
    w.stage = (tpc_cluster*)take((size_t)max_digits * sizeof(tpc_cluster));
    w.compact = (tpc_cluster*)take((size_t)max_clusters * sizeof(tpc_cluster));
    w.keyA = (uint64_t*)take((size_t)max_clusters * 8);
    w.keyB = (uint64_t*)take((size_t)max_clusters * 8);
    w.idxA = (uint32_t*)take((size_t)max_clusters * 4);
    w.idxB = (uint32_t*)take((size_t)max_clusters * 4);
    w.ghist = (uint32_t*)take((size_t)tiles * 256 * 4);
    w.ghist_part = (uint32_t*)take((ceil_div_u64(tiles * 256, 1024) + 1) * 4);
    w.line_start = (uint32_t*)take(((size_t)g.n_planes * g.LS + 2) * 4);
    w.line_cnt = (uint32_t*)take(((size_t)g.n_planes * g.LS + 2) * 4);
    w.line_desc = (unsigned long long*)take((ceil_div_u64((uint64_t)g.n_planes * g.LS + 2, 64) + 1) * 8);
    w.group_status = (tpc_cf_status*)take(sizeof(tpc_cf_status) * 32);
    w.sort_tmp = (tpc_digit*)take(sorted_only ? 0 : (size_t)max_digits * sizeof(tpc_digit));
    w.sort_top = (uint32_t*)take(1032 * 4);               // cursors of the digit sort's top-level buckets
    w.sort_part = (uint32_t*)take((ceil_div_u64((uint64_t)g.n_planes * g.LS + 2, 1024) + 4) * 4);
    if (ws) *ws = w;
    if (n_sort_tiles) *n_sort_tiles = (uint32_t)tiles;
    if (map_bytes) *map_bytes = mapb;
    return off;
}

static int cuda_fail(tpc_cf* h, cudaError_t e, const char* where)
{
    snprintf(g_last_cuda_msg, sizeof g_last_cuda_msg, "%s: %s", where, cudaGetErrorString(e));
    if (h) memcpy(h->cuda_msg, g_last_cuda_msg, sizeof h->cuda_msg);
    return TPC_CF_E_CUDA;
}

extern "C" size_t tpc_cf_workspace_bytes_ex(const tpc_cf_geometry* geom, uint64_t max_digits, uint64_t max_clusters,
                                            uint32_t ws_flags)
{
    Geo g;
    if (!geom || !geometry_to_geo(geom, &g)) return 0;
    if (max_digits >= (1ull << 32) || max_clusters >= (1ull << 32)) return 0;
    if (ws_flags & ~(uint32_t)TPC_CF_WS_SORTED_ONLY) return 0;
    return carve(g, max_digits, max_clusters, ws_flags, nullptr, nullptr, nullptr, nullptr);
}

extern "C" size_t tpc_cf_workspace_bytes(const tpc_cf_geometry* geom, uint64_t max_digits, uint64_t max_clusters)
{
    return tpc_cf_workspace_bytes_ex(geom, max_digits, max_clusters, 0u);
}

extern "C" int tpc_cf_create(tpc_cf** hp, const tpc_cf_geometry* geom, uint64_t max_digits, uint64_t max_clusters,
                             void* workspace, size_t workspace_bytes, void* stream)
{
    return tpc_cf_create_ex(hp, geom, max_digits, max_clusters, 0u, workspace, workspace_bytes, stream);
}

extern "C" int tpc_cf_create_ex(tpc_cf** hp, const tpc_cf_geometry* geom, uint64_t max_digits, uint64_t max_clusters,
                                uint32_t ws_flags, void* workspace, size_t workspace_bytes, void* stream)
{
    if (ws_flags & ~(uint32_t)TPC_CF_WS_SORTED_ONLY) return TPC_CF_E_PARAMS;
    if (!hp || !geom || !workspace) return TPC_CF_E_NULL;
    Geo g;
    if (!geometry_to_geo(geom, &g)) return TPC_CF_E_GEOMETRY;
    if (max_digits >= (1ull << 32) || max_clusters >= (1ull << 32)) return TPC_CF_E_CAPACITY;
    if (((uintptr_t)workspace & 255u) != 0) return TPC_CF_E_WORKSPACE;
    if (carve(g, max_digits, max_clusters, ws_flags, nullptr, nullptr, nullptr, nullptr) > workspace_bytes)
        return TPC_CF_E_WORKSPACE;
    tpc_cf* h = new (std::nothrow) tpc_cf;
    if (!h) return TPC_CF_E_NOMEM;
    memset(h, 0, sizeof *h);
    h->geo = g;
    h->max_digits = max_digits;
    h->max_clusters = max_clusters;
    h->ws_flags = ws_flags;
    carve(g, max_digits, max_clusters, ws_flags, (char*)workspace, &h->ws, &h->n_sort_tiles, &h->map_bytes);
    for (int i = 0; i < kProfSlots * 4; ++i) {
        cudaError_t e = cudaEventCreate(&h->ev[i / 4][i % 4]);
        if (e != cudaSuccess) { delete h; return cuda_fail(nullptr, e, "cudaEventCreate"); }
    }
    // the fused kernels use more than 48 KB of dynamic shared memory: a per-device attribute, set for this handle's device
    cudaError_t e = fused_pairs_set_attributes();
    if (e == cudaSuccess) e = fused_blocks_set_attributes();
    if (e == cudaSuccess) e = fused_lines_set_attributes();
    if (e == cudaSuccess) e = sort_set_attributes();
    // K0, once: the charge map starts zero; every run restores it (un-scatter).
    if (e == cudaSuccess && h->map_bytes) e = cudaMemsetAsync(h->ws.map, 0, h->map_bytes, (cudaStream_t)stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->ws.counters, 0, sizeof(Counters), (cudaStream_t)stream);
    if (e != cudaSuccess) {
        for (int i = 0; i < kProfSlots * 4; ++i) cudaEventDestroy(h->ev[i / 4][i % 4]);
        delete h;
        return cuda_fail(nullptr, e, "tpc_cf_create (kernel attributes / map zeroing)");
    }
    *hp = h;
    return TPC_CF_OK;
}

static int check_run_args(tpc_cf* h, const tpc_digit* digits, uint64_t n, const tpc_cf_geometry* geom,
                          const tpc_cf_params* params)
{
    if (!h || !geom || !params || (n && !digits)) return TPC_CF_E_NULL;
    Geo g;
    if (!geometry_to_geo(geom, &g) || !same_geometry(g, h->geo)) return TPC_CF_E_GEOMETRY;
    if (n > h->max_digits) return TPC_CF_E_CAPACITY;
    if (params->q_peak_min == 0) return TPC_CF_E_PARAMS;
    if (params->flags & ~(uint32_t)(TPC_CF_DIGITS_SORTED | TPC_CF_FORCE_GENERAL | TPC_CF_CLUSTER_FLAGS |
                                    TPC_CF_CUT_SINGLE_PAD | TPC_CF_CUT_SINGLE_TIME | TPC_CF_SHARE_CHARGE)) return TPC_CF_E_PARAMS;
    if (((uintptr_t)digits & 7u) != 0) return TPC_CF_E_NULL;
    return TPC_CF_OK;
}

extern "C" int tpc_cf_run(tpc_cf* h, const tpc_digit* digits, uint64_t n, const tpc_cf_geometry* geom,
                          const tpc_cf_params* params, tpc_cf_out* out)
{
    int rc = check_run_args(h, digits, n, geom, params);
    if (rc != TPC_CF_OK) return rc;
    if (!out || !out->status || (out->capacity && !out->clusters)) return TPC_CF_E_NULL;
    if (((uintptr_t)out->clusters & 15u) != 0 || ((uintptr_t)out->status & 7u) != 0) return TPC_CF_E_NULL;
    cudaStream_t st = (cudaStream_t)out->stream;
    const bool hint = (params->flags & TPC_CF_DIGITS_SORTED) != 0;
    const bool fused = hint && !(params->flags & TPC_CF_FORCE_GENERAL);
    if (!fused && (h->ws_flags & TPC_CF_WS_SORTED_ONLY)) return TPC_CF_E_PARAMS;   // no map, no sort buffer in this workspace
    // no promise about the order: sort the digits on the device, then the fused path (tpc_cf_sort.cu)
    const bool sortfuse = !hint && !(params->flags & TPC_CF_FORCE_GENERAL) && n > 0;
    const bool prof = h->profiling != 0;
    cudaEvent_t* ev = h->ev[h->run_index % kProfSlots];
    int k = 0;

    Variant var;
    var.q_tot_min = params->q_tot_min;
    var.q_saturation = params->q_saturation;
    var.vflags = params->flags & (TPC_CF_CLUSTER_FLAGS | TPC_CF_CUT_SINGLE_PAD | TPC_CF_CUT_SINGLE_TIME);
    var.active = (var.q_tot_min != 0u || var.vflags != 0u) ? 1u : 0u;
    const bool share = (params->flags & TPC_CF_SHARE_CHARGE) != 0;

    (void)cudaGetLastError();
    if (prof) cudaEventRecord(ev[0], st);
    cudaError_t e = cudaSuccess;
    if (!fused || n == 0) {       // (the fused path's index kernel zeroes the counters)
        e = cudaMemsetAsync(h->ws.counters, 0, sizeof(Counters), st);
        if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemsetAsync(counters)");
    }

    NvtxRange nv_run(fused ? "tpc_cf_run (fused path)" : sortfuse ? "tpc_cf_run (digit sort + fused path)" : "tpc_cf_run (general path)");
    if (fused || sortfuse) {
        // T3: (digit sort ->) line index -> fused smem kernel (scatter into smem lines, peak test, moments) -> compaction
        const tpc_digit* src = digits;
        if (sortfuse) {
            NvtxRange nv("K5 first: digit sort (partition by pad line, rank by time)");
            k += launch_sort_digits(h->geo, h->ws, digits, n, st);
            src = h->ws.sort_tmp;
        }
        int r;
        {
            NvtxRange nv("K0 K1 K2 K4: line index + fused kernel (clean, scatter, peaks, moments)");
            r = launch_fused_sorted(h->geo, h->ws, src, n, h->shape_n ? h->shape_n : h->shape_hint, params->q_peak_min,
                                    params->q_inner_gate, var, h->tun, sortfuse, st, prof ? ev[1] : nullptr, prof ? ev[2] : nullptr);
        }
        if (r < 0) return r;
        k += r;
        NvtxRange nv("K3 K5: scan + ordered copy + status");
        k += launch_compact_lines(h->geo, h->ws, out->clusters, out->capacity, out->status, n, sortfuse ? 2u : 3u, st);
        if (share) {
            NvtxRange nv6("K6: charge sharing between overlapping clusters (V4)");
            k += launch_share_charge(h->geo, h->ws, src, out->clusters, out->capacity, out->status, params->q_inner_gate,
                                     var.vflags, h->max_digits, st);
        }
    } else {
        // T1: K1 scatter -> K2+K4 digit-centric peaks + moments on the HBM map -> K3 compaction -> (K5 key sort)
        //     -> K0 un-scatter
        { NvtxRange nv("K1 K2 K4: scatter, peaks + moments on the map");
          k += launch_general_peaks(h->geo, h->ws, digits, n, params->q_peak_min, params->q_inner_gate, var, st,
                                    prof ? ev[1] : nullptr, prof ? ev[2] : nullptr); }
        { NvtxRange nv("K3: compaction");
          k += launch_compact(h->ws, n, out->clusters, out->capacity, h->max_clusters, hint ? 0 : 1, st); }
        if (!hint) { NvtxRange nv("K5: key sort"); k += launch_key_sort(h->ws, h->max_clusters, h->n_sort_tiles, out->clusters, out->capacity, st); }
        k += launch_finalize(h->ws, out->status, out->capacity, 1u, hint ? 1 : 0, n, h->max_clusters, st);
        if (share) {                  // (reads the map: ahead of the un-scatter)
            NvtxRange nv6("K6: charge sharing between overlapping clusters (V4)");
            k += launch_share_charge(h->geo, h->ws, nullptr, out->clusters, out->capacity, out->status,
                                     params->q_inner_gate, var.vflags, h->max_digits, st);
        }
        { NvtxRange nv("K0: un-scatter"); k += launch_unscatter(h->geo, h->ws, digits, n, st); }
    }
    if (prof) { cudaEventRecord(ev[3], st); ++h->run_index; }
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(h, e, "kernel launch");
    h->last_launches = k;
    h->last_kernel = g_last_kernel;
    return TPC_CF_OK;
}

static bool ensure_pipe(tpc_cf* h)
{
    if (h->pipe_ready) return true;
    bool ok = cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking) == cudaSuccess &&
              cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) == cudaSuccess;
    for (int i = 0; ok && i < kMaxGroups; ++i)
        ok = cudaEventCreateWithFlags(&h->ev_in[i], cudaEventDisableTiming) == cudaSuccess &&
             cudaEventCreateWithFlags(&h->ev_run[i], cudaEventDisableTiming) == cudaSuccess;
    ok = ok && cudaHostAlloc((void**)&h->pinned_status, sizeof(tpc_cf_status) * kMaxGroups, cudaHostAllocDefault) == cudaSuccess;
    if (!ok) { (void)cudaGetLastError(); return false; }    // leaks a few handles on a failing device; caller falls back
    h->pipe_ready = true;
    return true;
}

// first index in host digits [0, n) whose sector is >= s (digits promised sorted; terminates on any input)
static uint64_t host_lower_bound_sector(const tpc_digit* d, uint64_t n, uint32_t s)
{
    uint64_t lo = 0, hi = n;
    while (lo < hi) {
        const uint64_t mid = lo + ((hi - lo) >> 1);
        if (d[mid].sector < s) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// Sorted frames are pipelined over groups of whole sectors: the copy-in of group g+1 (stream s_in) overlaps the run of
// group g (caller's stream) and the copy-out of group g-1 (stream s_out).  Sectors are independent (R2), groups are in
// sector order, so the concatenated outputs are the frame's output.  Returns 1 if the frame was delivered, 0 if the
// caller must take the single-shot route (false promise, a group over its share of the capacity, CUDA hiccup in the
// pipeline set-up), < 0 on error.
static int run_host_pipelined(tpc_cf* h, const tpc_digit* host_digits, uint64_t n, const tpc_cf_geometry* geom,
                              const tpc_cf_params* params, tpc_digit* dev_digits, tpc_cluster* dev_clusters,
                              tpc_cluster* host_clusters, uint64_t capacity, tpc_cf_status* host_status,
                              cudaStream_t st, bool* digits_on_device)
{
    if (!ensure_pipe(h)) return 0;
    // group boundaries: sector-aligned, near equal digit counts
    uint64_t b[kMaxGroups + 1];
    int G = 0;
    b[0] = 0;
    const int want = (int)(geom->n_sectors < (uint32_t)kMaxGroups ? geom->n_sectors : (uint32_t)kMaxGroups);
    for (int g = 1; g < want; ++g) {
        const uint64_t probe = n * (uint64_t)g / (uint64_t)want;
        const uint64_t cut = host_lower_bound_sector(host_digits, n, host_digits[probe].sector);
        if (cut > b[G] && cut < n) b[++G] = cut;
    }
    b[++G] = n;
    if (G < 2) return 0;

    cudaError_t e = cudaEventRecord(h->ev_fork, st);                 // earlier work on the caller's stream comes first
    if (e == cudaSuccess) e = cudaStreamWaitEvent(h->s_in, h->ev_fork, 0);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(h->s_out, h->ev_fork, 0);
    for (int g = 0; e == cudaSuccess && g < G; ++g) {
        e = cudaMemcpyAsync(dev_digits + b[g], host_digits + b[g], (b[g + 1] - b[g]) * sizeof(tpc_digit),
                            cudaMemcpyHostToDevice, h->s_in);
        if (e == cudaSuccess) e = cudaEventRecord(h->ev_in[g], h->s_in);
    }
    if (e != cudaSuccess) return cuda_fail(h, e, "pipeline H2D");
    *digits_on_device = true;                                        // (once s_in has drained)
    uint64_t off[kMaxGroups + 1];
    off[0] = 0;
    for (int g = 0; g < G; ++g) {
        const uint64_t ng = b[g + 1] - b[g];
        const uint64_t cap = g + 1 < G ? (uint64_t)((double)capacity * ((double)ng / (double)n)) : capacity - off[g];
        off[g + 1] = off[g] + cap;
        e = cudaStreamWaitEvent(st, h->ev_in[g], 0);
        if (e != cudaSuccess) return cuda_fail(h, e, "pipeline wait");
        tpc_cf_out out = { dev_clusters + off[g], cap, h->ws.group_status + g, (void*)st };
        h->shape_n = n;
        const int rc = tpc_cf_run(h, dev_digits + b[g], ng, geom, params, &out);
        h->shape_n = 0;
        if (rc != TPC_CF_OK) { cudaStreamSynchronize(h->s_in); cudaStreamSynchronize(st); return rc; }
        e = cudaMemcpyAsync(h->pinned_status + g, h->ws.group_status + g, sizeof(tpc_cf_status), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaEventRecord(h->ev_run[g], st);
        if (e != cudaSuccess) return cuda_fail(h, e, "pipeline status");
    }
    tpc_cf_status tot;
    memset(&tot, 0, sizeof tot);
    tot.path = 3;
    bool redo = false;
    for (int g = 0; g < G; ++g) {
        e = cudaEventSynchronize(h->ev_run[g]);
        if (e != cudaSuccess) return cuda_fail(h, e, "pipeline sync");
        const tpc_cf_status s = h->pinned_status[g];
        if (s.path != 3 || s.overflow) redo = true;                  // false promise / group over its share
        if (redo) continue;
        if (s.n_clusters) {
            e = cudaMemcpyAsync(host_clusters + tot.n_clusters, dev_clusters + off[g], s.n_clusters * sizeof(tpc_cluster),
                                cudaMemcpyDeviceToHost, h->s_out);
            if (e != cudaSuccess) return cuda_fail(h, e, "pipeline D2H");
        }
        tot.n_clusters += s.n_clusters;
        tot.n_digits_used += s.n_digits_used;
        tot.n_bad_digits += s.n_bad_digits;
    }
    e = cudaStreamSynchronize(h->s_out);
    if (e == cudaSuccess) e = cudaStreamSynchronize(h->s_in);
    if (e != cudaSuccess) return cuda_fail(h, e, "pipeline drain");
    if (redo) return 0;
    *host_status = tot;
    return 1;
}

extern "C" int tpc_cf_run_host(tpc_cf* h, const tpc_digit* host_digits, uint64_t n, const tpc_cf_geometry* geom,
                               const tpc_cf_params* params, tpc_digit* dev_digits, tpc_cluster* dev_clusters,
                               tpc_cf_status* dev_status, tpc_cluster* host_clusters, uint64_t capacity,
                               tpc_cf_status* host_status, void* stream)
{
    if (!h || !params || !host_status || !dev_status || (n && (!host_digits || !dev_digits))) return TPC_CF_E_NULL;
    if (capacity && (!dev_clusters || !host_clusters)) return TPC_CF_E_NULL;
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaSuccess;
    bool on_device = false;
    const bool sorted_hint = (params->flags & TPC_CF_DIGITS_SORTED) && !(params->flags & TPC_CF_FORCE_GENERAL);
    if (sorted_hint && geom && geom->n_sectors >= 2 && n >= (1u << 22) && n <= h->max_digits && capacity >= 1024) {
        const int r = run_host_pipelined(h, host_digits, n, geom, params, dev_digits, dev_clusters, host_clusters,
                                         capacity, host_status, st, &on_device);
        if (r != 0) return r < 0 ? r : TPC_CF_OK;
    }
    if (n && !on_device) e = cudaMemcpyAsync(dev_digits, host_digits, n * sizeof(tpc_digit), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemcpyAsync(H2D digits)");
    tpc_cf_params prm = *params;
    for (int attempt = 0; attempt < 2; ++attempt) {
        tpc_cf_out out = { dev_clusters, capacity, dev_status, stream };
        int rc = tpc_cf_run(h, dev_digits, n, geom, &prm, &out);
        if (rc != TPC_CF_OK) return rc;
        e = cudaMemcpyAsync(host_status, dev_status, sizeof(tpc_cf_status), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(h, e, "status readback");
        if (host_status->path != 0 || (h->ws_flags & TPC_CF_WS_SORTED_ONLY)) break;   // (no general path to fall back on)
        prm.flags &= ~(uint32_t)TPC_CF_DIGITS_SORTED;   // the promise was false: rerun on the general path
    }
    uint64_t m = host_status->n_clusters < capacity ? host_status->n_clusters : capacity;
    if (m) {
        e = cudaMemcpyAsync(host_clusters, dev_clusters, m * sizeof(tpc_cluster), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(h, e, "cluster readback");
    }
    return TPC_CF_OK;
}

extern "C" int tpc_cf_debug_dense_plane(tpc_cf* h, const tpc_digit* digits, uint64_t n, uint32_t sector,
                                        uint32_t row, uint16_t* dense, void* stream)
{
    if (!h || !dense || (n && !digits)) return TPC_CF_E_NULL;
    if (n > h->max_digits) return TPC_CF_E_CAPACITY;
    if (sector >= h->geo.n_sectors || row >= h->geo.n_rows) return TPC_CF_E_GEOMETRY;
    if (h->ws_flags & TPC_CF_WS_SORTED_ONLY) return TPC_CF_E_PARAMS;
    cudaStream_t st = (cudaStream_t)stream;
    (void)cudaGetLastError();
    cudaMemsetAsync(h->ws.counters, 0, sizeof(Counters), st);
    launch_scatter_only(h->geo, h->ws, digits, n, st);
    launch_copy_plane(h->geo, h->ws, sector * h->geo.n_rows + row, h->geo.npads[row], dense, st);
    launch_unscatter(h->geo, h->ws, digits, n, st);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(h, e, "debug_dense_plane");
    return TPC_CF_OK;
}

extern "C" int tpc_cf_set_frame_digits(tpc_cf* h, uint64_t frame_digits)
{
    if (!h) return TPC_CF_E_NULL;
    h->shape_hint = frame_digits;
    return TPC_CF_OK;
}

extern "C" int tpc_cf_debug_set(tpc_cf* h, int key, int value)
{
    if (!h) return TPC_CF_E_NULL;
    if (value < 0) return TPC_CF_E_PARAMS;
    switch (key) {
    case TPC_CF_DEBUG_FUSED_KERNEL: if (value > 3) return TPC_CF_E_PARAMS; h->tun.fused_kernel = value; break;
    case TPC_CF_DEBUG_PASSES: h->tun.passes = value; break;
    case TPC_CF_DEBUG_BLOCK_POOL: h->tun.block_pool = value; break;
    case TPC_CF_DEBUG_SURV_CAP: h->tun.surv_cap = value; break;
    case TPC_CF_DEBUG_PADS_PER_UNIT: h->tun.pads_per_unit = value; break;
    case TPC_CF_DEBUG_CTAS_PER_SM: h->tun.ctas_per_sm = value; break;
    default: return TPC_CF_E_PARAMS;
    }
    return TPC_CF_OK;
}

extern "C" int tpc_cf_debug_scan_u32(tpc_cf* h, const uint32_t* in, uint32_t* out, uint64_t n, unsigned long long* total,
                                     void* stream)
{
    if (!h || (n && (!in || !out))) return TPC_CF_E_NULL;
    // partial sums in the handle's workspace (the cluster staging area is idle between runs)
    if ((ceil_div_u64(n, 1024) + 1) * 4 > h->max_digits * sizeof(tpc_cluster)) return TPC_CF_E_CAPACITY;
    (void)cudaGetLastError();
    launch_scan_u32(in, out, n, (uint32_t*)h->ws.stage, total, (cudaStream_t)stream);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(h, e, "debug_scan_u32");
    return TPC_CF_OK;
}

extern "C" int tpc_cf_last_launch_count(const tpc_cf* h) { return h ? h->last_launches : TPC_CF_E_NULL; }

extern "C" const char* tpc_cf_last_kernel(const tpc_cf* h) { return h && h->last_kernel ? h->last_kernel : ""; }

extern "C" int tpc_cf_set_profiling(tpc_cf* h, int on)
{
    if (!h) return TPC_CF_E_NULL;
    h->profiling = on ? 1 : 0;
    h->run_index = 0;
    return TPC_CF_OK;
}

extern "C" float tpc_cf_profile_ms(tpc_cf* h, uint32_t run, int which)
{
    if (!h || !h->profiling || run >= h->run_index || run + kProfSlots < h->run_index) return -1.f;
    cudaEvent_t* ev = h->ev[run % kProfSlots];
    float ms = -1.f;
    cudaError_t e;
    if (which == 0) { e = cudaEventSynchronize(ev[3]); if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ev[0], ev[3]); }
    else            { e = cudaEventSynchronize(ev[2]); if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ev[1], ev[2]); }
    if (e != cudaSuccess) { cuda_fail(h, e, "event timing"); return -1.f; }
    return ms;
}

extern "C" int tpc_cf_destroy(tpc_cf* h)
{
    if (!h) return TPC_CF_E_NULL;
    for (int i = 0; i < kProfSlots * 4; ++i) cudaEventDestroy(h->ev[i / 4][i % 4]);
    if (h->pipe_ready) {
        cudaStreamDestroy(h->s_in); cudaStreamDestroy(h->s_out);
        cudaEventDestroy(h->ev_fork); cudaEventDestroy(h->ev_join);
        for (int i = 0; i < kMaxGroups; ++i) { cudaEventDestroy(h->ev_in[i]); cudaEventDestroy(h->ev_run[i]); }
        cudaFreeHost(h->pinned_status);
    }
    delete h;
    return TPC_CF_OK;
}

extern "C" const char* tpc_cf_strerror(int code)
{
    switch (code) {
    case TPC_CF_OK: return "ok";
    case TPC_CF_E_NULL: return "required pointer is NULL or misaligned";
    case TPC_CF_E_GEOMETRY: return "invalid geometry, or geometry differs from create";
    case TPC_CF_E_CAPACITY: return "n exceeds max_digits, or a capacity is >= 2^32";
    case TPC_CF_E_WORKSPACE: return "workspace too small or not 256-byte aligned";
    case TPC_CF_E_PARAMS: return "invalid params (q_peak_min == 0, unknown flag bits, or a general-path run on a sorted-only workspace)";
    case TPC_CF_E_CUDA: return g_last_cuda_msg[0] ? g_last_cuda_msg : "CUDA error";
    case TPC_CF_E_NOMEM: return "host allocation failed";
    default: return "unknown error";
    }
}
