// S6: tracklet selector -- "selection of good tracks and final assignment of clusters to tracks dissolving
// ambiguities".  Reading: every cluster goes to the claiming tracklet with the most
// hits (ties: lowest candidate id); a tracklet keeps the hits it won and becomes a final track iff it keeps
// >= sel_min hits; final tracks are numbered in ascending candidate id.  Integer-only, so results are unique.
//
// Warp per tracklet (the row-indexed hit table of one tracklet is one coalesced 2*R-byte read); claim by a 32-bit
// atomicMax on the packed weight (nhits << 23 | inverted candidate id local to the sector instance); deterministic
// numbering through per-block counts + one scan + in-block prefix.
#include "tpc_common.cuh"

namespace tpc {

constexpr int kSelThreads = 256;
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kSelBlock = 64;  // tracklets per CTA work item
constexpr int kSelPerWarp = kSelBlock / kSelWarps;

struct TlView {
    int inst, first, last;
    uint32_t w;
    const uint16_t* rowhit;
    const int32_t* ro;
};

__device__ __forceinline__ bool load_tracklet(const DevGeom& g, int64_t c, const int32_t* __restrict__ row_offsets,
                                              const int32_t* __restrict__ tl_nhits,
                                              const int32_t* __restrict__ tl_rows,
                                              const int32_t* __restrict__ cand_slab,
                                              const int2* __restrict__ slab_part,
                                              const uint16_t* __restrict__ tl_rowhit, int64_t* counts, TlView& v) {
    const int nh = tl_nhits[c];
    if (nh == 0) return false;
    const int rows = tl_rows[c];
    v.first = rows & 0xff;
    v.last = (rows >> 8) & 0xff;
    v.inst = cand_slab[c] / g.R;
    const int64_t lcid = c - slab_part[(size_t)v.inst * g.R].y;  // candidate ordinal inside its sector instance
    if (lcid > 0x7FFFFF) atomicOr((unsigned long long*)&counts[5], 2ull);
    v.w = ((uint32_t)nh << 23) | (uint32_t)(0x7FFFFF - (lcid & 0x7FFFFF));
    v.rowhit = tl_rowhit + c * g.RP;
    v.ro = row_offsets + (size_t)v.inst * g.R;
    return true;
}

__global__ void __launch_bounds__(kSelThreads)
claim_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
             const int32_t* __restrict__ tl_nhits, const int32_t* __restrict__ tl_rows,
             const int32_t* __restrict__ cand_slab, const int2* __restrict__ slab_part,
             const uint16_t* __restrict__ tl_rowhit, uint32_t* __restrict__ claim, int64_t* __restrict__ counts,
             int64_t Cmax) {
    const int64_t n_cand = min(counts[1], Cmax);
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = (int64_t)blockIdx.x * kSelWarps + (threadIdx.x >> 5);
    for (int64_t c = warp0; c < n_cand; c += (int64_t)gridDim.x * kSelWarps) {
        TlView v;
        if (!load_tracklet(g, c, row_offsets, tl_nhits, tl_rows, cand_slab, slab_part, tl_rowhit, counts, v)) continue;
        for (int r = v.first + lane; r <= v.last; r += 32) {
            const uint16_t li = v.rowhit[r];
            if (li != kNoHit) atomicMax(&claim[v.ro[r] + li], v.w);
        }
    }
}

__global__ void __launch_bounds__(kSelThreads)
count_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
             const int32_t* __restrict__ tl_nhits, const int32_t* __restrict__ tl_rows,
             const int32_t* __restrict__ cand_slab, const int2* __restrict__ slab_part,
             const uint16_t* __restrict__ tl_rowhit, const uint32_t* __restrict__ claim,
             int32_t* __restrict__ tl_kept, int2* __restrict__ sel_part, int64_t* __restrict__ counts, int64_t Cmax) {
    __shared__ int s_cnt[3];
    const int64_t n_cand = min(counts[1], Cmax);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int64_t blk = blockIdx.x; blk * kSelBlock < n_cand; blk += gridDim.x) {
        if (threadIdx.x < 3) s_cnt[threadIdx.x] = 0;
        __syncthreads();
        int n_trk = 0, n_hit = 0, n_tl = 0;
        for (int i = 0; i < kSelPerWarp; i++) {
            const int64_t c = blk * kSelBlock + wid * kSelPerWarp + i;
            if (c >= n_cand) break;
            TlView v;
            int kept = 0;
            if (load_tracklet(g, c, row_offsets, tl_nhits, tl_rows, cand_slab, slab_part, tl_rowhit, counts, v)) {
                n_tl++;
                for (int r = v.first + lane; r <= v.last; r += 32) {
                    const uint16_t li = v.rowhit[r];
                    if (li != kNoHit && claim[v.ro[r] + li] == v.w) kept++;
                }
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) kept += __shfl_xor_sync(0xffffffffu, kept, d);
                if (kept < g.sel_min) kept = 0;
            }
            if (lane == 0) tl_kept[c] = kept;
            n_trk += kept > 0;
            n_hit += kept;
        }
        if (lane == 0) {
            atomicAdd(&s_cnt[0], n_trk);
            atomicAdd(&s_cnt[1], n_hit);
            atomicAdd(&s_cnt[2], n_tl);
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            sel_part[blk] = make_int2(s_cnt[0], s_cnt[1]);
            if (s_cnt[2]) atomicAdd((unsigned long long*)&counts[2], (unsigned long long)s_cnt[2]);
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kSelThreads)
write_tracks_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
                    const int32_t* __restrict__ tl_nhits, const int32_t* __restrict__ tl_rows,
                    const int32_t* __restrict__ cand_slab, const int2* __restrict__ slab_part,
                    const uint16_t* __restrict__ tl_rowhit, const uint32_t* __restrict__ claim,
                    const int32_t* __restrict__ tl_kept, const int2* __restrict__ sel_part,
                    const float* __restrict__ tl_par, const float* __restrict__ tl_cov,
                    const float* __restrict__ tl_chi2, const uint16_t* __restrict__ hit_idx,
                    int64_t* __restrict__ counts, int64_t Cmax, const SelectOut o) {
    __shared__ int s_kept[kSelBlock];
    __shared__ int2 s_off[kSelBlock];
    const int64_t n_cand = min(counts[1], Cmax);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int64_t blk = blockIdx.x; blk * kSelBlock < n_cand; blk += gridDim.x) {
        if (threadIdx.x < kSelBlock) {
            const int64_t c = blk * kSelBlock + threadIdx.x;
            s_kept[threadIdx.x] = c < n_cand ? tl_kept[c] : 0;
        }
        __syncthreads();
        if (wid == 0) {  // exclusive prefix over the 64 tracklets of the block (two per lane)
            const int k0 = s_kept[2 * lane], k1 = s_kept[2 * lane + 1];
            int t = (k0 > 0) + (k1 > 0), h = k0 + k1;
            int ti = t, hi = h;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int a = __shfl_up_sync(0xffffffffu, ti, d), b = __shfl_up_sync(0xffffffffu, hi, d);
                if (lane >= d) { ti += a; hi += b; }
            }
            s_off[2 * lane] = make_int2(ti - t, hi - h);
            s_off[2 * lane + 1] = make_int2(ti - t + (k0 > 0), hi - h + k0);
        }
        __syncthreads();
        const int2 base = sel_part[blk];
        for (int i = 0; i < kSelPerWarp; i++) {
            const int q = wid * kSelPerWarp + i;
            const int64_t c = blk * kSelBlock + q;
            if (c >= n_cand || s_kept[q] == 0) continue;
            const int64_t trk = (int64_t)base.x + s_off[q].x;
            const int64_t h0 = (int64_t)base.y + s_off[q].y;
            TlView v;
            load_tracklet(g, c, row_offsets, tl_nhits, tl_rows, cand_slab, slab_part, tl_rowhit, counts, v);
            const bool fits = trk < o.trk_capacity;
            if (fits) {
                if (o.trk_params && lane < 5) o.trk_params[trk * 5 + lane] = tl_par[c * 5 + lane];
                if (o.trk_cov && lane < 15) o.trk_cov[trk * 15 + lane] = tl_cov[c * 15 + lane];
                if (lane == 0) {
                    if (o.trk_chi2) o.trk_chi2[trk] = tl_chi2[c];
                    if (o.trk_xref) o.trk_xref[trk] = g.row_x[(tl_rows[c] >> 16) & 0xff];
                    if (o.trk_cand_id) o.trk_cand_id[trk] = (int32_t)c;
                    if (o.trk_nhits) o.trk_nhits[trk] = s_kept[q];
                    if (o.trk_sector) o.trk_sector[trk] = v.inst;
                    if (o.trk_hit_offset) o.trk_hit_offset[trk] = h0;
                }
            }
            int run = 0;
            for (int rb = v.first; rb <= v.last; rb += 32) {
                const int r = rb + lane;
                int gh = -1;
                if (r <= v.last) {
                    const uint16_t li = v.rowhit[r];
                    if (li != kNoHit) {
                        const int hh = v.ro[r] + li;  // sorted space; the outputs take the input-order index
                        if (claim[hh] == v.w) gh = v.ro[r] + (int)hit_idx[hh];
                    }
                }
                const unsigned m = __ballot_sync(0xffffffffu, gh >= 0);
                if (gh >= 0 && fits) {
                    const int64_t pos = h0 + run + __popc(m & ((1u << lane) - 1u));
                    if (o.trk_hits && pos < o.trk_hits_capacity) o.trk_hits[pos] = gh;
                    if (o.cluster_owner) o.cluster_owner[gh] = (int32_t)trk;
                }
                run += __popc(m);
            }
        }
        __syncthreads();
    }
}

__global__ void finalize_counts_kernel(const int64_t* __restrict__ counts, const SelectOut o) {
    if (threadIdx.x == 0) {
        if (o.trk_hit_offset && counts[3] <= o.trk_capacity) o.trk_hit_offset[counts[3]] = counts[4];
    }
    if (threadIdx.x < 16) o.counts[threadIdx.x] = counts[threadIdx.x];
}

// defined in k34_links_chains.cu
void launch_scan_int2(int2* part, const int64_t* m_dev, int64_t m_div, int64_t m_cap, int64_t m_host, int64_t* counts,
                      int c0, int c1, cudaStream_t s);

int launch_select(const DevGeom& g, const Workspace& w, const Problem& p, const SelectOut& o, cudaStream_t s) {
    int launches = 0;
    if (p.n_clusters > 0) {
        const int64_t blocks = div_up(w.Cmax, kSelBlock);
        const int grid_b = (int)(blocks < 148 * 16 ? blocks : 148 * 16);
        const int64_t warps = div_up(w.Cmax, kSelWarps);
        const int grid_w = (int)(warps < 148 * 16 ? warps : 148 * 16);
        claim_kernel<<<grid_w, kSelThreads, 0, s>>>(g, p.row_offsets, w.tl_nhits, w.tl_rows, w.cand_slab, w.slab_part,
                                                    w.tl_rowhit, w.claim, w.counts, w.Cmax);
        count_kernel<<<grid_b, kSelThreads, 0, s>>>(g, p.row_offsets, w.tl_nhits, w.tl_rows, w.cand_slab, w.slab_part,
                                                    w.tl_rowhit, w.claim, w.tl_kept, w.sel_part, w.counts, w.Cmax);
        launch_scan_int2(w.sel_part, w.counts + 1, kSelBlock, w.Cmax, 0, w.counts, 3, 4, s);
        write_tracks_kernel<<<grid_b, kSelThreads, 0, s>>>(g, p.row_offsets, w.tl_nhits, w.tl_rows, w.cand_slab,
                                                           w.slab_part, w.tl_rowhit, w.claim, w.tl_kept, w.sel_part,
                                                           w.tl_par, w.tl_cov, w.tl_chi2, w.hit_idx, w.counts, w.Cmax, o);
        launches += 4;
    }
    finalize_counts_kernel<<<1, 32, 0, s>>>(w.counts, o);
    return launches + 1;
}

// Parity/debug export: tracklet hit table as global cluster indices, rows as three ints.
__global__ void export_tracklets_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
                                        const int32_t* __restrict__ tl_nhits, const int32_t* __restrict__ tl_rows,
                                        const int32_t* __restrict__ cand_slab,
                                        const uint16_t* __restrict__ tl_rowhit,
                                        const uint16_t* __restrict__ hit_idx, const int64_t* __restrict__ counts,
                                        int64_t cap, int32_t* __restrict__ out_hits, int32_t* __restrict__ out_rows) {
    const int64_t n_cand = min(counts[1], cap);
    const int lane = threadIdx.x & 31;
    const int64_t warp0 = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    for (int64_t c = warp0; c < n_cand; c += (int64_t)gridDim.x * (blockDim.x >> 5)) {
        const int nh = tl_nhits[c];
        const int rows = tl_rows[c];
        const int first = rows & 0xff, last = (rows >> 8) & 0xff, ref = (rows >> 16) & 0xff;
        const int inst = cand_slab[c] / g.R;
        const int32_t* ro = row_offsets + (size_t)inst * g.R;
        if (out_rows && lane < 3) out_rows[c * 3 + lane] = nh ? (lane == 0 ? first : lane == 1 ? last : ref) : -1;
        if (out_hits)
            for (int r = lane; r < g.R; r += 32) {
                int gh = -1;
                if (nh && r >= first && r <= last) {
                    const uint16_t li = tl_rowhit[c * g.RP + r];
                    if (li != kNoHit) gh = ro[r] + (int)hit_idx[ro[r] + li];
                }
                out_hits[c * g.R + r] = gh;
            }
    }
}

int launch_export_tracklets(const DevGeom& g, const Workspace& w, const Problem& p, int32_t* tl_hits, int32_t* tl_rows,
                            int64_t cap, cudaStream_t s) {
    if (p.n_clusters == 0 || (!tl_hits && !tl_rows)) return 0;
    const int64_t c = cap < w.Cmax ? cap : w.Cmax;
    if (c <= 0) return 0;
    const int64_t warps = div_up(c, 8);
    const int grid = (int)(warps < 148 * 16 ? warps : 148 * 16);
    export_tracklets_kernel<<<grid, 256, 0, s>>>(g, p.row_offsets, w.tl_nhits, w.tl_rows, w.cand_slab, w.tl_rowhit,
                                                 w.hit_idx, w.counts, c, tl_hits, tl_rows);
    return 1;
}

}  // namespace tpc
