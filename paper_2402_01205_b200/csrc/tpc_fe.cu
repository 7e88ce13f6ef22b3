// tpc_fe.cu — TPC front-end filter "TPC-FE v1" (include/tpc_fe.h; step named in PAPER.md:57): common-mode correction,
// ion-tail cancellation and zero suppression of the raw, time-major ADC samples -> sorted tpc_digit records.
// Product code, sm_100a.  Shares nothing with oracle/tpc_fe_oracle.c: the definition text in the header is the only link.
//
// On the caller's stream:
//   k_fe_filter   the dense pass (HBM-bound by design: every raw sample is read exactly once).  Persistent CTAs, one
//                 (sector,row) plane at a time, one thread per pad.  The plane streams through a ring of kStages
//                 tiles of kTT time bins in shared memory; a tile is one contiguous piece of the time-major input and
//                 is fetched with one bulk copy (cp.async.bulk + mbarrier transaction count), kStages - 1 tiles ahead.
//                 Per tile: (1) a warp per time bin forms the quiet-pad sum and count in one packed accumulator and one
//                 warp reduction -> cm[t]; (2) every thread walks its pad through the tile's time bins with the tail
//                 state in a register, marks the kept bins in a 64-bit mask and overwrites their cells with q;
//                 (3) every pad line appends its kept (time, q) words to 32-record chunks of the plane's staging area; a
//                 warp scan hands out the chunks, a directory entry names a chunk's pad and first rank.  Per-line and
//                 per-warp counts at the end of the plane.
//   k_fe_scan     exclusive scan of the plane counts
//   k_fe_order    one CTA per plane: line offsets from the line counts, then a warp per chunk copies it (128 bytes in,
//                 256 bytes out) to out[plane offset + line offset + first rank ..]: ascending (sector,row,pad,time)
//                 without a sort; the status is written by the CTA that finishes last
#include <new>

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tpc_fe.h"

namespace tpcfe {

static constexpr int kTT = 64;          // time bins per tile (the kept-bin mask is 64 bits)
static constexpr int kStages = 2;       // tiles in the ring: kStages - 1 in flight ahead of the one in work
static constexpr int kSlack = 128;      // bytes after the ring: phase 1 may read up to 31 samples past a row's pitch
static constexpr int kChunk = 32;       // records per staging chunk (one 128-byte line)
static constexpr int kAccShift = 22;    // packed quiet-pad accumulator: count << 22 | sum (|sum| < 2^20)

struct Args {
    const uint16_t* raw;
    const uint16_t* ped4;
    const uint32_t* npads;      // [n_rows]
    uint32_t n_planes, n_rows, n_time, W;
    uint32_t zs, c, m, k, mul;  // zs_threshold, cm_quiet4, cm_min_pads, it_decay_shift, 1 << (14 - kappa) or 0
    uint32_t cpp;               // staging chunks per plane (a chunk = kChunk records of one pad line, consecutive ranks)
    uint32_t* temp;             // [n_planes][cpp][kChunk]: (time | q << 16)
    uint32_t* dir;              // [n_planes][cpp]: pad | (rank / kChunk) << 8 of the chunk
    uint32_t* line_cnt;         // [n_planes][W]
    uint32_t* warp_cnt;         // [n_planes][8]: kept samples of the pads of warp w (pads 32 w .. 32 w + 31)
    uint32_t* warp_chunks;      // [n_planes][8]: chunks opened by warp w
    uint32_t* flags;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}

__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// one contiguous piece of global memory -> shared memory, completion counted in bytes on the mbarrier
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, unsigned long long* bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// NW = warps per CTA = ceil(W / 32); WC = W when it is known at compile time (immediate offsets), else 0
template <int NW, int WC>
__global__ void __launch_bounds__(NW * 32) k_fe_filter(const Args a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    uint16_t* tiles = (uint16_t*)smem;                    // [kStages][kTT * W]
    __shared__ __align__(8) unsigned long long s_bar[kStages];
    __shared__ __align__(16) int s_cm[2][kTT];
    __shared__ int s_mul;

    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t W = WC ? (uint32_t)WC : a.W, T = a.n_time;
    const uint32_t tile_elems = kTT * W;
    const uint32_t tpp = (T + kTT - 1) / kTT;                                   // tiles per plane
    const uint32_t my_planes = blockIdx.x < a.n_planes ? (a.n_planes - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    const uint32_t total_tiles = my_planes * tpp;

    if (tid == 0) {
        s_mul = (int)a.mul;
        for (int s = 0; s < kStages; s++) mbar_init(&s_bar[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    auto issue = [&](uint32_t m) {                                              // thread 0 only
        const uint32_t lp = m / tpp, tl = m - lp * tpp;
        const uint32_t plane = blockIdx.x + lp * gridDim.x;
        const uint32_t t0 = tl * kTT;
        const uint32_t nt = min((uint32_t)kTT, T - t0);
        const uint16_t* src = a.raw + ((size_t)plane * T + t0) * W;
        bulk_load(tiles + (size_t)(m % kStages) * tile_elems, src, nt * W * 2u, &s_bar[m % kStages]);
    };
    if (tid == 0)
        for (uint32_t m = 0; m < (uint32_t)(kStages - 1) && m < total_tiles; m++) issue(m);

    const uint32_t c2 = 2u * a.c;
    const uint32_t capw = a.cpp / NW;                                           // staging chunks per warp and plane
    const int kk = (int)a.k, zs = (int)a.zs;
    // read back from shared memory so that it lives in a register (else the compiler reloads it from the constant bank,
    // predicated, once per sample)
    const int mul = *(volatile int*)&s_mul;
    const uint32_t bias = (1u << kAccShift) - a.c;
    uint32_t n = 0;                                                             // tile sequence number of this CTA
    for (uint32_t lp = 0; lp < my_planes; lp++) {
        const uint32_t plane = blockIdx.x + lp * gridDim.x;
        const uint32_t P = a.npads[plane % a.n_rows];
        const bool active = tid < P;
        const uint16_t* ped = a.ped4 + (size_t)plane * W;
        const int pedneg2 = active ? 2 - (int)ped[tid] : 0;                     // z + 2 = 4 raw + (2 - ped) - cm + tail
        // phase-1 view: lane handles pads lane + 32 g
        uint32_t pedq[NW];
#pragma unroll
        for (int g = 0; g < NW; g++) {
            const uint32_t pad = lane + 32u * g;
            pedq[g] = pad < P ? a.c - (uint32_t)ped[min(pad, W - 1)] : 0x40000000u;         // beyond the row: never quiet
        }
        int S = 0;
        uint32_t cnt = 0;       // kept samples of this pad line so far (rank of the next one)
        uint32_t wpos = 0;      // kept samples of this warp's pads so far (same value in every lane)
        uint32_t wchunks = 0;   // chunks opened by this warp so far (same value in every lane)
        uint32_t cur = 0;       // the chunk this pad line is filling
        uint32_t* wtemp = a.temp + ((size_t)plane * a.cpp + (size_t)warp * capw) * kChunk;
        uint32_t* wdir = a.dir + (size_t)plane * a.cpp + (size_t)warp * capw;

        for (uint32_t tl = 0; tl < tpp; tl++, n++) {
            const uint32_t t0 = tl * kTT;
            const uint32_t nt = min((uint32_t)kTT, T - t0);
            uint16_t* tile = tiles + (size_t)(n % kStages) * tile_elems;
            int* cmv = s_cm[n & 1];
            mbar_wait(&s_bar[n % kStages], (n / kStages) & 1u);

            // ---- (1) common mode of every time bin of the tile: warp `warp` takes bins warp, warp + NW, ...; lane l
            // keeps the packed sum of the warp's l-th bin and turns it into cm when 32 bins (or the tile) are done
            {
                auto flush = [&](uint32_t b_first, uint32_t n_bins, int mine) {
                    if (lane < n_bins) {
                        const uint32_t i = warp + (b_first + lane) * NW;
                        const int nq = (mine + (1 << (kAccShift - 1))) >> kAccShift;
                        const int s = mine - (nq << kAccShift);
                        int cm = 0;
                        if (nq >= (int)a.m && nq > 0) {
                            const int num = 2 * s + nq, den = 2 * nq;
                            cm = num / den;
                            if (num - cm * den < 0) cm -= 1;                             // floor
                        }
                        cmv[i] = cm;
                    }
                };
                uint32_t b = 0;
                int mine = 0;
                for (uint32_t i = warp; i < nt; i += NW, b++) {
                    const uint16_t* row = tile + i * W + lane;
                    int acc = 0;
#pragma unroll
                    for (int g = 0; g < NW; g++) {
                        const uint32_t xb = (uint32_t)row[32 * g] * 4u + pedq[g];        // x + c
                        acc += xb <= c2 ? (int)(xb + bias) : 0;                          // x + 2^22
                    }
                    acc = __reduce_add_sync(0xffffffffu, acc);
                    if (lane == (b & 31u)) mine = acc;
                    if ((b & 31u) == 31u) { flush(b - 31u, 32u, mine); mine = 0; }
                }
                if (b & 31u) flush(b & ~31u, b & 31u, mine);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // this thread's q stores into tile n - 1
            __syncthreads();
            // every thread is past tile n - 1: its stage is free for tile n + kStages - 1
            if (tid == 0 && n + kStages - 1 < total_tiles) issue(n + kStages - 1);

            // ---- (2) the pad's walk through the tile
            uint32_t mlo = 0, mhi = 0;
            if (active) {
                uint16_t* cell = tile + tid;
                if (nt == (uint32_t)kTT) {
#pragma unroll
                    for (int i4 = 0; i4 < kTT; i4 += 4) {
                        const int4 cm4 = *(const int4*)(cmv + i4);
                        const int cma[4] = {cm4.x, cm4.y, cm4.z, cm4.w};
#pragma unroll
                        for (int u = 0; u < 4; u++) {
                            const int i = i4 + u;
                            const int base = (int)cell[i * W] * 4 + (pedneg2 - cma[u]);     // independent of S
                            const int q = min((base + (S >> 12)) >> 2, 65535);
                            S -= S >> kk;
                            if (q >= zs) {
                                S += q * mul;
                                cell[i * W] = (uint16_t)q;
                                if (i < 32) mlo |= 1u << i; else mhi |= 1u << (i - 32);
                            }
                        }
                    }
                } else {
                    for (uint32_t i = 0; i < nt; i++) {
                        const int base = (int)cell[i * W] * 4 + (pedneg2 - cmv[i]);
                        const int q = min((base + (S >> 12)) >> 2, 65535);
                        S -= S >> kk;
                        if (q >= zs) {
                            S += q * mul;
                            cell[i * W] = (uint16_t)q;
                            if (i < 32) mlo |= 1u << i; else mhi |= 1u << (i - 32);
                        }
                    }
                }
            }

            // ---- (3) stage the tile's records: a pad line fills chunks of kChunk records (consecutive ranks) taken from
            // the warp's part of the plane's staging area; a warp scan hands out the chunks the lanes open in this tile
            // (no block barrier; k_fe_order copies chunk by chunk, coalesced, to where the line's ranks belong)
            {
                const uint32_t c = __popc(mlo) + __popc(mhi);
                const uint32_t opened = ((cnt + c + kChunk - 1) / kChunk) - ((cnt + kChunk - 1) / kChunk);
                uint32_t incl = opened;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
                    if (lane >= (uint32_t)d) incl += v;
                }
                uint32_t next_new = wchunks + incl - opened;
                wchunks += __shfl_sync(0xffffffffu, incl, 31);
                wpos += (uint32_t)__reduce_add_sync(0xffffffffu, c);
                if (c) {
                    const uint32_t cell_addr = smem_u32(tile + tid);
                    uint32_t rank = cnt;
                    auto put = [&](uint32_t i) {
                        uint32_t q;
                        asm volatile("ld.shared.u16 %0, [%1];" : "=r"(q) : "r"(cell_addr + i * (W * 2u)));
                        if ((rank & (kChunk - 1)) == 0u) {
                            cur = next_new++;
                            if (cur < capw) wdir[cur] = tid | ((rank / kChunk) << 8);
                        }
                        if (cur < capw) wtemp[cur * kChunk + (rank & (kChunk - 1))] = (t0 + i) | (q << 16);
                        rank++;
                    };
                    while (mlo) { put(__ffs(mlo) - 1); mlo &= mlo - 1; }
                    while (mhi) { put(__ffs(mhi) + 31); mhi &= mhi - 1; }
                    cnt = rank;
                }
            }
        }
        if (tid < W) a.line_cnt[(size_t)plane * W + tid] = cnt;
        if (lane == 0) {
            a.warp_cnt[(size_t)plane * 8 + warp] = wpos;
            a.warp_chunks[(size_t)plane * 8 + warp] = wchunks;
            if (wchunks > capw) atomicOr(a.flags, (uint32_t)TPC_FE_OVF_PLANE);
        }
        if (tid >= NW && tid < 8) {
            a.warp_cnt[(size_t)plane * 8 + tid] = 0;
            a.warp_chunks[(size_t)plane * 8 + tid] = 0;
        }
    }
}

// exclusive scan of the plane counts (one CTA), status
__global__ void __launch_bounds__(1024) k_fe_scan(const uint32_t* warp_cnt, uint32_t n_planes, uint64_t* plane_off,
                                                  uint32_t* flags)
{
    __shared__ uint64_t s_w[32];
    __shared__ uint64_t s_carry;
    const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (uint32_t b = 0; b < n_planes; b += 1024) {
        const uint32_t i = b + tid;
        uint64_t v = 0;
        if (i < n_planes) {
            const uint4 a4 = ((const uint4*)warp_cnt)[2 * (size_t)i], b4 = ((const uint4*)warp_cnt)[2 * (size_t)i + 1];
            v = (uint64_t)a4.x + a4.y + a4.z + a4.w + b4.x + b4.y + b4.z + b4.w;
        }
        uint64_t incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint64_t u = __shfl_up_sync(0xffffffffu, incl, d);
            if (lane >= (uint32_t)d) incl += u;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        uint64_t before = s_carry;
        for (uint32_t w = 0; w < warp; w++) before += s_w[w];
        if (i < n_planes) plane_off[i] = before + incl - v;
        __syncthreads();
        if (tid == 1023) s_carry = before + incl;
        __syncthreads();
    }
    if (tid == 0) *(uint64_t*)(flags + 2) = s_carry;       // total; the status is written by the last CTA of k_fe_order
}

// one CTA per plane: staged chunks -> their place in the sorted output (a warp per chunk: 128 bytes in, 256 bytes out)
__global__ void __launch_bounds__(256) k_fe_order(const uint32_t* temp_all, const uint32_t* dir_all, uint32_t cpp,
                                                  const uint32_t* line_cnt, const uint32_t* warp_chunks,
                                                  const uint64_t* plane_off, uint32_t W, uint32_t n_rows, uint2* out,
                                                  uint64_t capacity, uint32_t* flags, tpc_fe_status* status)
{
    __shared__ uint32_t s_off[256];
    __shared__ uint32_t s_cnt[256];
    __shared__ uint32_t s_w[8];
    const uint32_t plane = blockIdx.x, tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
    const uint32_t v = tid < W ? line_cnt[(size_t)plane * W + tid] : 0;
    uint32_t incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= (uint32_t)d) incl += u;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    uint32_t before = 0;
    for (uint32_t w = 0; w < warp; w++) before += s_w[w];
    s_off[tid] = before + incl - v;
    s_cnt[tid] = v;
    __syncthreads();
    const uint64_t base = plane_off[plane];
    const uint32_t head = (plane / n_rows) | ((plane % n_rows) << 8);
    const uint32_t nw = (W + 31) / 32, capw = cpp / nw;
    for (uint32_t w = 0; w < nw; w++) {
        const uint32_t n = min(warp_chunks[(size_t)plane * 8 + w], capw);
        const uint32_t* temp = temp_all + ((size_t)plane * cpp + (size_t)w * capw) * kChunk;
        const uint32_t* dir = dir_all + (size_t)plane * cpp + (size_t)w * capw;
        for (uint32_t ch = warp; ch < n; ch += 8) {
            const uint32_t e = dir[ch];
            const uint32_t pad = e & 255u, first = (e >> 8) * kChunk;          // rank of the chunk's first record
            const uint32_t cnt = s_cnt[pad];
            if (first + lane < cnt) {
                const uint64_t dst = base + s_off[pad] + first + lane;
                if (dst < capacity) out[dst] = make_uint2(head | (pad << 16), temp[ch * kChunk + lane]);
            }
        }
    }
    // the status is written last: by the CTA that finishes last
    __threadfence();
    __syncthreads();
    if (tid == 0 && atomicAdd(flags + 1, 1u) == gridDim.x - 1) {
        const uint64_t total = *(const volatile uint64_t*)(flags + 2);
        status->n_digits = total;
        status->overflow = *(const volatile uint32_t*)flags | (total > capacity ? (uint32_t)TPC_FE_OVF_OUTPUT : 0u);
        status->rsv = 0;
    }
}

}  // namespace tpcfe

using namespace tpcfe;

struct tpc_fe {
    uint32_t n_sectors, n_rows, max_pads, n_time, W, n_planes;
    uint64_t cap;
    uint32_t* temp;
    uint32_t* dir;
    uint32_t* line_cnt;
    uint32_t* warp_cnt;
    uint32_t* warp_chunks;
    uint64_t* plane_off;
    uint32_t* npads;
    uint32_t* flags;
    uint32_t grid, smem;
    int last_launches;
    int profiling, have_pair;
    cudaEvent_t ev0, ev1;
};

static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static size_t carve(uint32_t n_planes, uint32_t n_rows, uint32_t W, uint64_t cap, char* base, tpc_fe* e)
{
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off += align256(bytes); return base ? base + o : (char*)nullptr; };
    char* p;
    p = take(256);                                   if (e) e->flags = (uint32_t*)p;
    p = take(4ull * n_rows);                         if (e) e->npads = (uint32_t*)p;
    p = take(32ull * n_planes);                      if (e) e->warp_cnt = (uint32_t*)p;
    p = take(32ull * n_planes);                      if (e) e->warp_chunks = (uint32_t*)p;
    p = take(4ull * n_planes * (cap / kChunk));      if (e) e->dir = (uint32_t*)p;
    p = take(8ull * n_planes);                       if (e) e->plane_off = (uint64_t*)p;
    p = take(4ull * n_planes * W);                   if (e) e->line_cnt = (uint32_t*)p;
    p = take(4ull * n_planes * (cap / kChunk) * kChunk); if (e) e->temp = (uint32_t*)p;
    return off;
}

static bool geometry_ok(const tpc_cf_geometry* g)
{
    if (g->n_sectors == 0 || g->n_sectors > 256 || g->n_rows == 0 || g->n_rows > 256 || g->max_pads == 0 ||
        g->max_pads > 255 || g->n_time == 0 || g->n_time > 65535) return false;
    if (g->npads)
        for (uint32_t r = 0; r < g->n_rows; r++)
            if (g->npads[r] == 0 || g->npads[r] > g->max_pads) return false;
    return true;
}

extern "C" uint32_t tpc_fe_pad_stride(uint32_t max_pads) { return (max_pads + 7u) / 8u * 8u; }

extern "C" size_t tpc_fe_workspace_bytes(const tpc_cf_geometry* g, uint64_t max_digits_per_plane)
{
    if (!g || !geometry_ok(g) || max_digits_per_plane == 0 || max_digits_per_plane >= (1ull << 32)) return 0;
    return carve(g->n_sectors * g->n_rows, g->n_rows, tpc_fe_pad_stride(g->max_pads), max_digits_per_plane, nullptr,
                 nullptr);
}

template <int NW, int WC>
static void setup_kernel(tpc_fe* e)
{
    int dev = 0, sms = 148, per_sm = 1;
    if (cudaFuncSetAttribute(k_fe_filter<NW, WC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)e->smem) != cudaSuccess ||
        cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_fe_filter<NW, WC>, NW * 32, e->smem) != cudaSuccess) {
        cudaGetLastError();      // no device (host-only tests): the launch will report it
        sms = 148; per_sm = 1;
    }
    if (per_sm < 1) per_sm = 1;
    e->grid = (uint32_t)(sms * per_sm);
}

extern "C" int tpc_fe_create(tpc_fe** h, const tpc_cf_geometry* g, uint64_t max_digits_per_plane, void* workspace,
                             size_t workspace_bytes)
{
    if (!h || !g || !workspace) return TPC_CF_E_NULL;
    if (!geometry_ok(g)) return TPC_CF_E_GEOMETRY;
    if (max_digits_per_plane == 0 || max_digits_per_plane >= (1ull << 32)) return TPC_CF_E_CAPACITY;
    const uint32_t W = tpc_fe_pad_stride(g->max_pads), n_planes = g->n_sectors * g->n_rows;
    if (((uintptr_t)workspace & 255u) != 0 ||
        workspace_bytes < carve(n_planes, g->n_rows, W, max_digits_per_plane, nullptr, nullptr))
        return TPC_CF_E_WORKSPACE;
    tpc_fe* e = new (std::nothrow) tpc_fe;
    if (!e) return TPC_CF_E_NOMEM;
    e->n_sectors = g->n_sectors; e->n_rows = g->n_rows; e->max_pads = g->max_pads; e->n_time = g->n_time;
    e->W = W; e->n_planes = n_planes; e->cap = max_digits_per_plane; e->last_launches = 0;
    e->profiling = 0; e->have_pair = 0; e->ev0 = nullptr; e->ev1 = nullptr;
    carve(n_planes, g->n_rows, W, max_digits_per_plane, (char*)workspace, e);
    uint32_t np[256];
    for (uint32_t r = 0; r < g->n_rows; r++) np[r] = g->npads ? g->npads[r] : g->max_pads;
    if (cudaMemcpy(e->npads, np, 4ull * g->n_rows, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        delete e;
        return TPC_CF_E_CUDA;
    }
    e->smem = (uint32_t)(kStages * kTT * W * 2u) + kSlack;
    switch ((W + 31) / 32) {
        case 1: setup_kernel<1, 0>(e); break;
        case 2: setup_kernel<2, 0>(e); break;
        case 3: setup_kernel<3, 0>(e); break;
        case 4: setup_kernel<4, 0>(e); break;
        case 5: if (W == 144) setup_kernel<5, 144>(e); else setup_kernel<5, 0>(e); break;
        case 6: setup_kernel<6, 0>(e); break;
        case 7: setup_kernel<7, 0>(e); break;
        default: setup_kernel<8, 0>(e); break;
    }
    *h = e;
    return TPC_CF_OK;
}

extern "C" int tpc_fe_run(tpc_fe* h, const uint16_t* raw, const uint16_t* ped4, const tpc_fe_params* p, tpc_digit* out,
                          uint64_t capacity, tpc_fe_status* status, void* stream)
{
    if (!h || !raw || !ped4 || !p || !status || (!out && capacity)) return TPC_CF_E_NULL;
    const int k = p->it_decay_shift, j = p->it_kappa_shift;
    if (p->zs_threshold < 1 || p->cm_quiet4 > 4095 || p->cm_min_pads < 1 || k < 1 || k > 15 ||
        (j != 0 && (j < k || j > 14))) return TPC_CF_E_PARAMS;
    if (((uintptr_t)raw & 15u) != 0 || ((uintptr_t)out & 7u) != 0) return TPC_CF_E_WORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    Args a;
    a.raw = raw; a.ped4 = ped4; a.npads = h->npads;
    a.n_planes = h->n_planes; a.n_rows = h->n_rows; a.n_time = h->n_time; a.W = h->W;
    a.zs = p->zs_threshold; a.c = p->cm_quiet4; a.m = p->cm_min_pads; a.k = (uint32_t)k;
    a.mul = j ? 1u << (14 - j) : 0u;
    a.cpp = (uint32_t)(h->cap / kChunk); a.temp = h->temp; a.dir = h->dir; a.line_cnt = h->line_cnt;
    a.warp_cnt = h->warp_cnt; a.warp_chunks = h->warp_chunks; a.flags = h->flags;
    cudaMemsetAsync(h->flags, 0, 16, st);
    const uint32_t grid = h->grid < h->n_planes ? h->grid : h->n_planes;
    if (h->profiling) cudaEventRecord(h->ev0, st);
    switch ((h->W + 31) / 32) {
        case 1: k_fe_filter<1, 0><<<grid, 32, h->smem, st>>>(a); break;
        case 2: k_fe_filter<2, 0><<<grid, 64, h->smem, st>>>(a); break;
        case 3: k_fe_filter<3, 0><<<grid, 96, h->smem, st>>>(a); break;
        case 4: k_fe_filter<4, 0><<<grid, 128, h->smem, st>>>(a); break;
        case 5:
            if (h->W == 144) k_fe_filter<5, 144><<<grid, 160, h->smem, st>>>(a);
            else k_fe_filter<5, 0><<<grid, 160, h->smem, st>>>(a);
            break;
        case 6: k_fe_filter<6, 0><<<grid, 192, h->smem, st>>>(a); break;
        case 7: k_fe_filter<7, 0><<<grid, 224, h->smem, st>>>(a); break;
        default: k_fe_filter<8, 0><<<grid, 256, h->smem, st>>>(a); break;
    }
    if (h->profiling) { cudaEventRecord(h->ev1, st); h->have_pair = 1; }
    k_fe_scan<<<1, 1024, 0, st>>>(h->warp_cnt, h->n_planes, h->plane_off, h->flags);
    k_fe_order<<<h->n_planes, 256, 0, st>>>(h->temp, h->dir, (uint32_t)(h->cap / kChunk), h->line_cnt, h->warp_chunks, h->plane_off, h->W,
                                            h->n_rows, (uint2*)out, capacity, h->flags, status);
    h->last_launches = 3;
    return cudaGetLastError() == cudaSuccess ? TPC_CF_OK : TPC_CF_E_CUDA;
}

extern "C" int tpc_fe_last_launch_count(const tpc_fe* h) { return h ? h->last_launches : 0; }

extern "C" int tpc_fe_set_profiling(tpc_fe* h, int on)
{
    if (!h) return TPC_CF_E_NULL;
    if (on && !h->ev0) {
        if (cudaEventCreate(&h->ev0) != cudaSuccess || cudaEventCreate(&h->ev1) != cudaSuccess) {
            cudaGetLastError();
            return TPC_CF_E_CUDA;
        }
    }
    h->profiling = on ? 1 : 0;
    if (!on) h->have_pair = 0;
    return TPC_CF_OK;
}

extern "C" float tpc_fe_profile_ms(tpc_fe* h)
{
    if (!h || !h->have_pair) return -1.0f;
    float ms = -1.0f;
    if (cudaEventSynchronize(h->ev1) != cudaSuccess || cudaEventElapsedTime(&ms, h->ev0, h->ev1) != cudaSuccess) {
        cudaGetLastError();
        return -1.0f;
    }
    return ms;
}

extern "C" int tpc_fe_destroy(tpc_fe* h)
{
    if (!h) return TPC_CF_E_NULL;
    if (h->ev0) cudaEventDestroy(h->ev0);
    if (h->ev1) cudaEventDestroy(h->ev1);
    delete h;
    return TPC_CF_OK;
}
