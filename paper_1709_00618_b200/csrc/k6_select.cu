// S6: tracklet selector -- "selection of good tracks and final assignment of clusters to tracks dissolving
// ambiguities".  Reading: every cluster goes to the claiming tracklet with the most
// hits (ties: lowest candidate id); a tracklet keeps the hits it won and becomes a final track iff it keeps
// >= sel_min hits; final tracks are numbered in ascending candidate id.  Integer-only, so results are unique.
//
// claim + mark (one CTA per sector instance, shared memory): one 32-bit atomicMax of the packed weight (nhits << 23 |
// inverted candidate ordinal inside the sector instance) per attached hit, then per hit the winner tracklet from
// the claim word -> the row's bit in the winner's kept-row mask.  (Round 1 did both on global memory: 473 M scattered
// L2 reductions at 88 % of the L2's throughput, 2.9 ms; in shared memory 1.5 ms.)
// Everything after it is HIT- or tracklet-centric streaming:
//   count     per tracklet: kept = popcount(mask), tracks/hits per block of 256 tracklets, then one scan
//   finalize  per tracklet: track index and first hit position (deterministic: ascending candidate id), track record
//   write     per hit: owner and the track's hit list entry (rank = kept rows below, from the mask)
#include <mutex>

#include "tpc_common.cuh"

namespace tpc {

constexpr int kSelThreads = 256;
constexpr int kSelBlock = kSelThreads;  // tracklets per CTA in the tracklet-centric passes
constexpr int kHitThreads = 256;        // hit-centric passes: one WARP per (sector instance, pad row)
constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ int64_t winner_of(uint32_t w, int64_t cand_base) {
    return cand_base + (int64_t)(0x7FFFFFu - (w & 0x7FFFFFu));
}

// claim + mark for ONE SECTOR INSTANCE per CTA, in shared memory.  An instance's clusters are claimed only by its
// own tracklets, and both the claim words (4 B per cluster, ~130 KB) and the kept-row masks (20 B per tracklet,
// ~30 KB) of one instance fit in an SM's shared memory: the ~4.6 claims per kept hit become shared-memory atomics
// instead of scattered L2 reductions (the separate kernels ran at 88 % of the L2's throughput: 473 M REDs), and the
// winners' mask bits are set in shared memory too.  The final claim words and masks go to global memory coalesced,
// once.  An instance too large for the shared memory (dense events) takes the same code on the global arrays.
constexpr int kInstThreads = 1024;

template <bool kShared>
__device__ __forceinline__ void claim_mark_instance(const DevGeom& g, const int32_t* __restrict__ s_ro,
                                                    const int32_t* __restrict__ tl_nhits,
                                                    const int32_t* __restrict__ tl_rows,
                                                    const uint16_t* __restrict__ tl_rowhit, int64_t c_lo, int n_c,
                                                    uint32_t* claim_w, uint32_t* mask_w, int mask_stride) {
    // claim_w[i] = claim word of the instance's hit i (sorted position - first hit of the instance; s_ro holds the
    // row offsets relative to it); mask_w[k * mask_stride + q] = word q of the kept-row mask of its tracklet k.
    // The row tables of the instance's tracklets are one contiguous array (RP entries each): the CTA streams it in
    // 8-byte pieces (4 rows), consecutive threads on consecutive pieces.
    const int quads = g.RP / 4;
    const uint2* tab = reinterpret_cast<const uint2*>(tl_rowhit + (size_t)c_lo * g.RP);
    constexpr int kU = 4;  // independent 8-byte pieces per thread in flight (the phase is bound by memory parallelism)
    // piece q = tracklet q / quads, rows 4 * (q % quads) ...; the pair is advanced incrementally (no division per piece)
    const int n_items = n_c * quads;  // < 2^31: n_c <= 2^23 / ... in practice a few thousand
    const int k_step = kInstThreads / quads, r_step = kInstThreads - k_step * quads;
    int kq = (int)threadIdx.x / quads, rem = (int)threadIdx.x - kq * quads;
    for (int q0 = threadIdx.x; q0 < n_items; q0 += kU * kInstThreads) {
        uint2 v[kU];
        int k[kU], rq[kU], nh[kU], rows[kU];
#pragma unroll
        for (int u = 0; u < kU; u++) {
            const int q = q0 + u * kInstThreads;
            k[u] = -1;
            if (q < n_items) {
                k[u] = kq;
                rq[u] = 4 * rem;
                v[u] = __ldcs(&tab[q]);
                nh[u] = tl_nhits[c_lo + kq];
                rows[u] = tl_rows[c_lo + kq];
            }
            kq += k_step;
            rem += r_step;
            if (rem >= quads) { rem -= quads; kq++; }
        }
#pragma unroll
        for (int u = 0; u < kU; u++) {
            if (k[u] < 0 || nh[u] <= 0) continue;
            const int first = rows[u] & 0xff, last = (rows[u] >> 8) & 0xff;
            const uint32_t w = ((uint32_t)nh[u] << 23) | (uint32_t)(0x7FFFFF - k[u]);
            const uint32_t li[4] = {v[u].x & 0xffffu, v[u].x >> 16, v[u].y & 0xffffu, v[u].y >> 16};
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const int r = rq[u] + j;
                if (r >= first && r <= last && li[j] != kNoHit) atomicMax(&claim_w[s_ro[r] + (int)li[j]], w);
            }
        }
    }
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, n_warps = kInstThreads / 32;
    for (int r = wid; r < g.R; r += n_warps) {  // mark: one warp per pad row
        const int b = s_ro[r], n = s_ro[r + 1] - b;
        const uint32_t bit = 1u << (r & 31);
        for (int i = lane; i < n; i += 32) {
            const uint32_t w = claim_w[b + i];
            if (w) atomicOr(&mask_w[(size_t)(0x7FFFFFu - (w & 0x7FFFFFu)) * mask_stride + (r >> 5)], bit);
        }
    }
}

__global__ void __launch_bounds__(kInstThreads, 1)
claim_mark_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
                  const int32_t* __restrict__ tl_nhits, const int32_t* __restrict__ tl_rows,
                  const int2* __restrict__ slab_part, const uint16_t* __restrict__ tl_rowhit,
                  uint32_t* __restrict__ claim, uint32_t* __restrict__ tl_sel, const int64_t* __restrict__ counts,
                  int64_t Cmax, int smem_words) {
    extern __shared__ __align__(16) uint32_t s_mem[];
    __shared__ int32_t s_ro[kMaxRows + 1];  // row offsets of the instance relative to its first hit
    const int inst = blockIdx.x;
    const int32_t* ro = row_offsets + (size_t)inst * g.R;
    const int hit0 = ro[0], n_hits = ro[g.R] - hit0;
    for (int r = threadIdx.x; r <= g.R; r += kInstThreads) s_ro[r] = ro[r] - hit0;
    const int64_t n_cand = min(counts[1], Cmax);
    const int64_t c_lo = min((int64_t)slab_part[(size_t)inst * g.R].y, n_cand);
    const int64_t c_hi = min((int64_t)slab_part[(size_t)(inst + 1) * g.R].y, n_cand);
    const int n_c = (int)(c_hi - c_lo);
    if (n_c <= 0 || n_hits <= 0) return;  // claim words and masks stay zero (initialised by S3/S4 and S5); uniform
    const int words = g.sel_words;
    if ((int64_t)n_hits + (int64_t)n_c * words <= smem_words) {
        uint32_t* claim_s = s_mem;
        uint32_t* mask_s = s_mem + n_hits;
        for (int i = threadIdx.x; i < n_hits + n_c * words; i += kInstThreads) s_mem[i] = 0u;
        __syncthreads();
        claim_mark_instance<true>(g, s_ro, tl_nhits, tl_rows, tl_rowhit, c_lo, n_c, claim_s, mask_s, words);
        __syncthreads();
        for (int i = threadIdx.x; i < n_hits; i += kInstThreads) claim[hit0 + i] = claim_s[i];
        for (int i = threadIdx.x; i < n_c * words; i += kInstThreads) {
            const int k = i / words, q = i - k * words;
            tl_sel[(size_t)(c_lo + k) * g.sel_stride + q] = mask_s[i];
        }
    } else {  // does not fit: the same passes on the global arrays (zeroed by the earlier stages)
        __syncthreads();
        claim_mark_instance<false>(g, s_ro, tl_nhits, tl_rows, tl_rowhit, c_lo, n_c, claim + hit0,
                                   tl_sel + (size_t)c_lo * g.sel_stride, g.sel_stride);
    }
}

// kept hits of tracklet c from its mask (0 if below sel_min)
__device__ __forceinline__ int kept_of(const DevGeom& g, const uint32_t* __restrict__ tl_sel, int64_t c) {
    const uint4* rec = reinterpret_cast<const uint4*>(tl_sel + c * g.sel_stride);
    int kept = 0;
    for (int q = 0; q < g.sel_words; q += 4) {  // words past sel_words inside the last uint4 are masked below
        const uint4 v = rec[q >> 2];
        kept += __popc(v.x);
        if (q + 1 < g.sel_words) kept += __popc(v.y);
        if (q + 2 < g.sel_words) kept += __popc(v.z);
        if (q + 3 < g.sel_words) kept += __popc(v.w);
    }
    return kept < g.sel_min ? 0 : kept;
}

__global__ void __launch_bounds__(kSelThreads)
count_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ tl_nhits,
             const uint32_t* __restrict__ tl_sel, int2* __restrict__ sel_part, int64_t* __restrict__ counts,
             int64_t Cmax) {
    __shared__ int s_cnt[3];
    const int64_t n_cand = min(counts[1], Cmax);
    const int lane = threadIdx.x & 31;
    for (int64_t blk = blockIdx.x; blk * kSelBlock < n_cand; blk += gridDim.x) {
        if (threadIdx.x < 3) s_cnt[threadIdx.x] = 0;
        __syncthreads();
        const int64_t c = blk * kSelBlock + threadIdx.x;
        int kept = 0, have = 0;
        if (c < n_cand && tl_nhits[c] > 0) {
            have = 1;
            kept = kept_of(g, tl_sel, c);
        }
        const int n_trk = __reduce_add_sync(kFull, kept > 0 ? 1 : 0);
        const int n_hit = __reduce_add_sync(kFull, kept);
        const int n_tl = __reduce_add_sync(kFull, have);
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

struct FinalIn {
    const int32_t* tl_nhits;
    const int32_t* tl_rows;
    const int32_t* cand_slab;
    const float* tl_par;
    const float* tl_cov;
    const float* tl_chi2;
    const int2* sel_part;
    uint32_t* tl_sel;
    int64_t* counts;
    int64_t Cmax;
    int32_t* trk_cand;  // [Tmax] workspace copy of the track -> candidate map (phase 2)
    int64_t Tmax;
};

__global__ void __launch_bounds__(kSelThreads)
finalize_tracks_kernel(const __grid_constant__ DevGeom g, const FinalIn a, const SelectOut o) {
    __shared__ int2 s_warp[kSelThreads / 32];
    const int64_t n_cand = min(a.counts[1], a.Cmax);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int64_t blk = blockIdx.x; blk * kSelBlock < n_cand; blk += gridDim.x) {
        const int64_t c = blk * kSelBlock + threadIdx.x;
        int kept = 0;
        if (c < n_cand && a.tl_nhits[c] > 0) kept = kept_of(g, a.tl_sel, c);
        // exclusive prefix of (tracks, hits) inside the block: warp scan + warp totals
        const int t = kept > 0 ? 1 : 0;
        int ti = t, hi = kept;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int x = __shfl_up_sync(kFull, ti, d), y = __shfl_up_sync(kFull, hi, d);
            if (lane >= d) { ti += x; hi += y; }
        }
        if (lane == 31) s_warp[wid] = make_int2(ti, hi);
        __syncthreads();
        int2 off = a.sel_part[blk];
        for (int k = 0; k < wid; k++) { off.x += s_warp[k].x; off.y += s_warp[k].y; }
        __syncthreads();
        if (c >= n_cand) continue;
        const int64_t trk = (int64_t)off.x + ti - t;
        const int64_t h0 = (int64_t)off.y + hi - kept;
        const bool is_trk = kept > 0 && trk < o.trk_capacity;
        uint32_t* rec = a.tl_sel + c * g.sel_stride;
        rec[g.sel_words] = is_trk ? (uint32_t)trk : 0xFFFFFFFFu;
        rec[g.sel_words + 1] = (uint32_t)h0;
        if (kept > 0 && trk < a.Tmax) a.trk_cand[trk] = (int32_t)c;
        if (!is_trk) continue;
        const int rows = a.tl_rows[c];
        if (o.trk_params)
#pragma unroll
            for (int q = 0; q < 5; q++) o.trk_params[trk * 5 + q] = a.tl_par[c * 5 + q];
        if (o.trk_cov)
#pragma unroll
            for (int q = 0; q < 15; q++) o.trk_cov[trk * 15 + q] = a.tl_cov[c * 15 + q];
        if (o.trk_chi2) o.trk_chi2[trk] = a.tl_chi2[c];
        if (o.trk_xref) o.trk_xref[trk] = g.row_x[(rows >> 16) & 0xff];
        if (o.trk_cand_id) o.trk_cand_id[trk] = (int32_t)c;
        if (o.trk_nhits) o.trk_nhits[trk] = kept;
        if (o.trk_sector) o.trk_sector[trk] = a.cand_slab[c] / g.R;
        if (o.trk_hit_offset) o.trk_hit_offset[trk] = h0;
    }
}

__global__ void __launch_bounds__(kHitThreads)
write_hits_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
                  const int2* __restrict__ slab_part, const uint32_t* __restrict__ claim,
                  const uint32_t* __restrict__ tl_sel, const uint16_t* __restrict__ hit_idx, const SelectOut o,
                  int n_slabs) {
    const int slab = blockIdx.x * (kHitThreads / 32) + (threadIdx.x >> 5);  // one warp per slab
    if (slab >= n_slabs) return;
    const int inst = slab / g.R, r = slab - inst * g.R;
    const int base = row_offsets[slab], n = min(row_offsets[slab + 1] - base, 65535);
    if (n == 0) return;
    const int64_t cand_base = slab_part[(size_t)inst * g.R].y;
    const int wq = r >> 5;
    const uint32_t below = (1u << (r & 31)) - 1u;
    for (int i = threadIdx.x & 31; i < n; i += 32) {
        const uint32_t w = claim[base + i];
        if (!w) continue;
        const uint32_t* rec = tl_sel + winner_of(w, cand_base) * g.sel_stride;
        const uint32_t trk = rec[g.sel_words];
        if (trk == 0xFFFFFFFFu) continue;  // the winner is not a final track: the hit stays unassigned
        int rank = __popc(rec[wq] & below);
        for (int q = 0; q < wq; q++) rank += __popc(rec[q]);
        const int gi = base + (int)hit_idx[base + i];  // sorted space -> input-order index
        if (o.cluster_owner) o.cluster_owner[gi] = (int32_t)trk;
        const int64_t pos = (int64_t)rec[g.sel_words + 1] + rank;
        if (o.trk_hits && pos < o.trk_hits_capacity) o.trk_hits[pos] = gi;
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
        const int slabs = p.n_inst * g.R;
        const int64_t blocks = div_up(w.Cmax, kSelBlock);
        const int grid = (int)(blocks < 148 * 8 ? blocks : 148 * 8);
        const int hgrid = div_up(slabs, kHitThreads / 32);
        {
            // the opt-in shared-memory size is a property of (kernel, device): cached per device ordinal, set up by
            // whichever host thread launches on that device first
            static std::mutex mu;
            static int smem_by_dev[kMaxDeviceOrdinals] = {};
            int dev = 0;
            cudaGetDevice(&dev);
            dev = dev >= 0 && dev < kMaxDeviceOrdinals ? dev : 0;
            int smem_bytes;
            {
                std::lock_guard<std::mutex> lock(mu);
                if (!smem_by_dev[dev]) {
                    int max_optin = 0;
                    cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
                    smem_by_dev[dev] = (max_optin > 0 ? max_optin : 48 * 1024) - 2048;  // room for the static arrays
                    cudaFuncSetAttribute(claim_mark_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         smem_by_dev[dev]);
                }
                smem_bytes = smem_by_dev[dev];
            }
            claim_mark_kernel<<<p.n_inst, kInstThreads, smem_bytes, s>>>(g, p.row_offsets, w.tl_nhits, w.tl_rows,
                                                                         w.slab_part, w.tl_rowhit, w.claim, w.tl_sel,
                                                                         w.counts, w.Cmax, smem_bytes / 4);
        }
        count_kernel<<<grid, kSelThreads, 0, s>>>(g, w.tl_nhits, w.tl_sel, w.sel_part, w.counts, w.Cmax);
        launch_scan_int2(w.sel_part, w.counts + 1, kSelBlock, w.Cmax, 0, w.counts, 3, 4, s);
        const FinalIn a{w.tl_nhits, w.tl_rows, w.cand_slab, w.tl_par, w.tl_cov, w.tl_chi2, w.sel_part, w.tl_sel,
                        w.counts,   w.Cmax,    w.trk_cand,  w.Tmax};
        finalize_tracks_kernel<<<grid, kSelThreads, 0, s>>>(g, a, o);
        write_hits_kernel<<<hgrid, kHitThreads, 0, s>>>(g, p.row_offsets, w.slab_part, w.claim, w.tl_sel, w.hit_idx, o,
                                                        slabs);
        launches += 5;
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
