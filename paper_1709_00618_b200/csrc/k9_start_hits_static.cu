// tpc_start_hits_static: the start-hit list of S4 for callers that have no way to allocate device memory.
//
// Who that is.  tpc_track_sectors keeps its intermediate arrays in a workspace the caller allocates.  Some callers
// cannot allocate at all: a reconstruction component that runs inside a host framework which reserved the whole GPU
// at start-up and hands every component fixed input/output buffers and nothing else; a plug-in in an online loop
// where cudaMalloc is off limits because it synchronises the whole device and stalls the other components sharing
// it; code that was only lent a stream.  Such a caller that already holds the cleaned links of S3 (from an earlier
// stage, from another device, from a file) still needs the start hits in ascending order, and the ordered
// compaction that produces them needs memory of its own: one status word per tile of the input.  Here that memory
// is a file-scope __device__ array inside the library, so the call needs no workspace, no tracker handle and no
// allocation of any kind.
//
// The operation is S4's first half ("the Cellular Automaton ... concatenates these links to form track
// candidates": a candidate begins at a start hit): hit h is a start hit iff it has a cleaned up-link and no cleaned
// down-link.  The result equals `start_hits` / counts[0] of tpc_track_sectors on the same links, element by element.
//
// How it differs from the regular path (k34_links_chains.cu: per-slab counts, a scan kernel, a ranked write): ONE
// kernel, a single pass.  CTAs take tiles of 2,048 hits in ticket order, publish their count, and find the number of
// start hits before their tile by looking back over the status words of the earlier tiles (aggregate or inclusive
// prefix, value and state in one 64-bit word so that no fence is needed).  A CTA only ever waits for tiles with a
// smaller ticket, whose CTAs are already running, so the wait always ends.
//
// The scratch array is shared by every call in the process on that device and keeps the last call's contents: the
// ticket and the status words the call will use are zeroed on the caller's stream before the kernel.  Two calls that
// overlap on the GPU (different streams, or different host threads) therefore race on it; issue them on one stream
// or order them with events.
#include <mutex>
#include <string>

#include "../../include/tpc_tracker.h"
#include "tpc_common.cuh"
#include "tracker_handle.cuh"

namespace tpc {

constexpr int kSsThreads = 256;
constexpr int kSsItems = 8;                       // consecutive hits per thread
constexpr int kSsTile = kSsThreads * kSsItems;    // 2,048 hits per CTA
constexpr int64_t kSsMaxHits = TPC_STATIC_MAX_CLUSTERS;
constexpr int kSsMaxTiles = (int)(kSsMaxHits / kSsTile);  // 65,536
constexpr int kSsHeader = 32;                     // word 0 = ticket counter; the status words start 256 bytes in
static_assert(kSsMaxHits % kSsTile == 0, "the limit is a whole number of tiles");

// 8 * (32 + 65,536) bytes = 512.25 KB, held by every GPU that loads the library until the process exits.
// In HOST code this name is only a stand-in for the symbol, not a device address: the address a kernel can use comes
// from cudaGetSymbolAddress (scratch_for_current_device below).
static __device__ __align__(256) unsigned long long g_start_hits_scratch[kSsHeader + kSsMaxTiles];

constexpr unsigned long long kStAggregate = 1ull << 32, kStInclusive = 2ull << 32;

__global__ void __launch_bounds__(kSsThreads)
start_hits_static_kernel(const int32_t* __restrict__ link_up, const int32_t* __restrict__ link_dn, int64_t n,
                         int32_t* __restrict__ start_hits, int64_t cap, int64_t* __restrict__ n_start,
                         unsigned long long* scratch, int n_tiles) {
    __shared__ int s_tile;
    __shared__ uint32_t s_warp[kSsThreads / 32];
    __shared__ uint32_t s_excl;
    if (threadIdx.x == 0) s_tile = (int)atomicAdd(&scratch[0], 1ull);  // tiles in ticket order, not blockIdx order
    __syncthreads();
    const int tile = s_tile;
    volatile unsigned long long* status = scratch + kSsHeader;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t i0 = (int64_t)tile * kSsTile + (int64_t)threadIdx.x * kSsItems;

    // bit q of mask: hit i0 + q is a start hit (cleaned up-link, no cleaned down-link)
    uint32_t mask = 0;
    const bool aligned = ((reinterpret_cast<uintptr_t>(link_up) | reinterpret_cast<uintptr_t>(link_dn)) & 15) == 0;
    if (aligned && i0 + kSsItems <= n) {
        const int4 u0 = __ldg(reinterpret_cast<const int4*>(link_up + i0));
        const int4 u1 = __ldg(reinterpret_cast<const int4*>(link_up + i0) + 1);
        const int4 d0 = __ldg(reinterpret_cast<const int4*>(link_dn + i0));
        const int4 d1 = __ldg(reinterpret_cast<const int4*>(link_dn + i0) + 1);
        const int32_t u[kSsItems] = {u0.x, u0.y, u0.z, u0.w, u1.x, u1.y, u1.z, u1.w};
        const int32_t d[kSsItems] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
#pragma unroll
        for (int q = 0; q < kSsItems; q++) mask |= (u[q] >= 0 && d[q] < 0) ? (1u << q) : 0u;
    } else {
#pragma unroll
        for (int q = 0; q < kSsItems; q++)
            if (i0 + q < n && __ldg(&link_up[i0 + q]) >= 0 && __ldg(&link_dn[i0 + q]) < 0) mask |= 1u << q;
    }

    // start hits of this tile before this thread
    const uint32_t cnt = __popc(mask);
    uint32_t incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t o = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += o;
    }
    if (lane == 31) s_warp[wid] = incl;
    __syncthreads();
    uint32_t before = 0, total = 0;
#pragma unroll
    for (int k = 0; k < kSsThreads / 32; k++) {
        const uint32_t w = s_warp[k];
        if (k < wid) before += w;
        total += w;
    }

    // start hits before this tile: warp 0 looks back over the earlier tiles, 32 status words at a time
    if (wid == 0) {
        uint32_t excl = 0;
        if (tile == 0) {
            if (lane == 0) status[0] = kStInclusive | total;
        } else {
            if (lane == 0) status[tile] = kStAggregate | total;
            int look = tile - 1;
            while (true) {
                const int idx = look - lane;  // lanes past tile 0 read as "inclusive prefix 0"
                unsigned long long w;
                uint32_t st;
                while (true) {
                    w = kStInclusive;
                    if (idx >= 0) w = status[idx];
                    st = (uint32_t)(w >> 32);
                    if (!__any_sync(0xffffffffu, st == 0)) break;  // an earlier tile has not published yet
                    __nanosleep(40);
                }
                const unsigned has_incl = __ballot_sync(0xffffffffu, st == 2);
                const int first = has_incl ? __ffs(has_incl) - 1 : 31;  // nearest tile with an inclusive prefix
                const uint32_t v = __reduce_add_sync(0xffffffffu, lane <= first ? (uint32_t)w : 0u);
                excl += v;
                if (has_incl) break;
                look -= 32;
            }
            if (lane == 0) status[tile] = kStInclusive | (unsigned long long)(excl + total);
        }
        if (lane == 0) s_excl = excl;
    }
    __syncthreads();

    int64_t pos = (int64_t)s_excl + before + (incl - cnt);
#pragma unroll
    for (int q = 0; q < kSsItems; q++) {
        if (mask & (1u << q)) {
            if (pos < cap) start_hits[pos] = (int32_t)(i0 + q);
            pos++;
        }
    }
    if (tile == n_tiles - 1 && threadIdx.x == 0) *n_start = (int64_t)s_excl + total;  // required count, also on overflow
}

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_ss_mutex;
unsigned long long* g_ss_ptr[kMaxDevices] = {};  // device address of g_start_hits_scratch, per device ordinal

// Once per device, with that device current: ask the runtime where the array lives on THIS device.
cudaError_t scratch_for_current_device(unsigned long long** out, int* dev_out) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *dev_out = dev;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_ss_mutex);
    if (!g_ss_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_start_hits_scratch);
        if (e != cudaSuccess) return e;
        g_ss_ptr[dev] = static_cast<unsigned long long*>(p);
    }
    *out = g_ss_ptr[dev];
    return cudaSuccess;
}
}  // namespace

}  // namespace tpc

extern "C" int tpc_start_hits_static(const int32_t* link_up, const int32_t* link_dn, int64_t n_clusters,
                                     int32_t* start_hits, int64_t start_capacity, int64_t* n_start, void* cuda_stream) {
    using namespace tpc;
    if (n_clusters < 0 || start_capacity < 0 || !n_start || (n_clusters > 0 && (!link_up || !link_dn)) ||
        (start_capacity > 0 && !start_hits)) {
        tpc_set_handleless_error("tpc_start_hits_static: NULL or negative argument");
        return TPC_ERR_ARG;
    }
    if (n_clusters > kSsMaxHits) {
        tpc_set_handleless_error("tpc_start_hits_static: n_clusters = " + std::to_string(n_clusters) +
                                 " is beyond TPC_STATIC_MAX_CLUSTERS = " + std::to_string(kSsMaxHits) +
                                 ", the size the library's built-in scratch array was compiled for; split the input "
                                 "or use tpc_track_sectors with a workspace");
        return TPC_ERR_LIMIT;
    }
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    unsigned long long* scratch = nullptr;
    int dev = 0;
    cudaError_t e = scratch_for_current_device(&scratch, &dev);
    if (e == cudaSuccess) {
        const int n_tiles = (int)((n_clusters + kSsTile - 1) / kSsTile);
        if (n_tiles == 0) {
            e = cudaMemsetAsync(n_start, 0, sizeof(int64_t), s);
        } else {
            // the array still holds the previous call's ticket and status words: zero the part this call uses
            e = cudaMemsetAsync(scratch, 0, sizeof(unsigned long long) * (size_t)(kSsHeader + n_tiles), s);
            if (e == cudaSuccess) {
                start_hits_static_kernel<<<n_tiles, kSsThreads, 0, s>>>(link_up, link_dn, n_clusters, start_hits,
                                                                        start_capacity, n_start, scratch, n_tiles);
                e = cudaGetLastError();
            }
        }
    }
    if (e != cudaSuccess) {
        tpc_set_handleless_error(std::string("tpc_start_hits_static: CUDA: ") + cudaGetErrorString(e));
        return TPC_ERR_CUDA;
    }
    return TPC_OK;
}
