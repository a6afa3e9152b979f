// S3: neighbour cleaning (keep only mutual links; BASELINE.json north_star), fused into the first pass of
// S4: start hits + concatenation of links into track candidates "of usually 4 to 10 TPC hits" (Fig. 1b).
// All integer work; results are unique, so they must equal the oracle bit for bit.
//
// Deterministic compaction without atomics-ordered output: candidates are numbered in ascending global index of
// their start hit by (1) per-slab counts, (2) one exclusive scan over the S*R slab counts, (3) a ballot/popc
// ranking inside each slab CTA.
#include "tpc_common.cuh"

namespace tpc {

constexpr int kChainThreads = 128;
constexpr int kScanThreads = 1024;

// S3 + S4 pass 1, fused (SURVEY.md 8(d) budgets S3 with its neighbours; the raw links were written, read
// back, cleaned, written again and read a third time).  Per hit: the cleaned links are computed on the fly from the
// raw arrays -- cu = up_raw[h] if dn_raw[up_raw[h]] == h, cd likewise (reading S3: mutual links only) -- only the
// cleaned up-link is materialised (the S5 fit kernel walks it), plus the flags (bit0 start hit, bit1 candidate), the
// per-slab counts and the selector's claim word.  A start hit's chain is walked on the raw arrays with the same
// mutuality test, because the cleaned links of later rows may not have been written yet by their warps.
// One WARP per (instance,row) slab: a slab is ~200 hits and a short chain of dependent loads, so what bounds this
// pass is how many slabs an SM has in flight -- 64 with a warp each against 16 with a 128-thread CTA each -- and a
// warp needs no barrier.
__global__ void __launch_bounds__(kChainThreads)
clean_flags_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
                   const int32_t* __restrict__ up_raw, const int32_t* __restrict__ dn_raw, int32_t* __restrict__ up,
                   uint32_t* __restrict__ claim, uint8_t* __restrict__ flags, int2* __restrict__ slab_part,
                   int n_slabs) {
    const int slab = blockIdx.x * (kChainThreads / 32) + (threadIdx.x >> 5);
    if (slab >= n_slabs) return;
    const int lane = threadIdx.x & 31;
    const int base = row_offsets[slab], n = row_offsets[slab + 1] - base;
    int ns = 0, nc = 0;
    for (int i = lane; i < n; i += 32) {
        const int h = base + i;
        const int32_t u = up_raw[h], d = dn_raw[h];
        const int32_t cu = (u >= 0 && __ldg(&dn_raw[u]) == h) ? u : -1;
        const bool has_cd = d >= 0 && __ldg(&up_raw[d]) == h;
        up[h] = cu;
        claim[h] = 0u;
        uint8_t f = 0;
        if (cu >= 0 && !has_cd) {
            f = 1;
            int len = 2;  // h and cu
            int x = cu;
            while (len < g.cand_min) {
                const int nx = __ldg(&up_raw[x]);
                if (nx < 0 || __ldg(&dn_raw[nx]) != x) { x = -1; break; }
                x = nx;
                len++;
            }
            if (x >= 0 && len >= g.cand_min) f = 3;
        }
        flags[h] = f;
        ns += f & 1;
        nc += f >> 1;
    }
    ns = __reduce_add_sync(0xffffffffu, ns);
    nc = __reduce_add_sync(0xffffffffu, nc);
    if (lane == 0) slab_part[slab] = make_int2(ns, nc);
}

// Exclusive scan of int2 partials by ONE CTA (m is a few thousand to a few hundred thousand entries); entry m
// receives the totals, which also go to counts[c0], counts[c1].
__global__ void __launch_bounds__(kScanThreads)
scan_int2_kernel(int2* __restrict__ part, const int64_t* __restrict__ m_dev, int64_t m_div, int64_t m_cap,
                 int64_t m_host, int64_t* __restrict__ counts, int c0, int c1) {
    __shared__ int2 s_warp[kScanThreads / 32];
    __shared__ int2 s_carry;
    // number of entries: host value, or ceil(min(*m_dev, m_cap) / m_div) when m_dev is given (S6: device-side count)
    const int64_t m = m_dev ? (min(*m_dev, m_cap) + m_div - 1) / m_div : m_host;
    if (threadIdx.x == 0) s_carry = make_int2(0, 0);
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    constexpr int kPer = 4;  // consecutive entries per thread and round
    for (int64_t start = 0; start < m; start += kScanThreads * kPer) {
        const int64_t i0 = start + (int64_t)threadIdx.x * kPer;
        int2 v[kPer];
        int2 sum = make_int2(0, 0);
#pragma unroll
        for (int q = 0; q < kPer; q++) {
            v[q] = i0 + q < m ? part[i0 + q] : make_int2(0, 0);
            sum.x += v[q].x;
            sum.y += v[q].y;
        }
        int2 incl = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int a = __shfl_up_sync(0xffffffffu, incl.x, d), b = __shfl_up_sync(0xffffffffu, incl.y, d);
            if (lane >= d) { incl.x += a; incl.y += b; }
        }
        if (lane == 31) s_warp[wid] = incl;
        __syncthreads();
        int2 off = s_carry;
        for (int k = 0; k < wid; k++) { off.x += s_warp[k].x; off.y += s_warp[k].y; }
        int2 run = make_int2(off.x + incl.x - sum.x, off.y + incl.y - sum.y);
#pragma unroll
        for (int q = 0; q < kPer; q++) {
            if (i0 + q < m) part[i0 + q] = run;
            run.x += v[q].x;
            run.y += v[q].y;
        }
        __syncthreads();
        if (threadIdx.x == kScanThreads - 1) s_carry = run;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        part[m] = s_carry;
        counts[c0] = s_carry.x;
        counts[c1] = s_carry.y;
    }
}

// S4 pass 2: ranked write of the start hits and of the candidates' start positions.  Links and flags live in sorted
// space, but start hits and candidates are numbered in ascending INPUT index of the start hit, so the
// CTA walks its row in input order (through S1's inverse permutation hit_pos) and ranks with ballot/popc prefixes.
// The candidate's hit list itself (the first <= 10 chain hits) is read off the links by the S5 fit kernel, one thread
// per candidate, where the walk runs at full lane occupancy.
__global__ void __launch_bounds__(kChainThreads)
chain_write_kernel(const int32_t* __restrict__ row_offsets, const uint16_t* __restrict__ hit_pos,
                   const uint8_t* __restrict__ flags, const int2* __restrict__ slab_part,
                   int32_t* __restrict__ start_hits, int64_t start_cap, int32_t* __restrict__ cand_start,
                   int32_t* __restrict__ cand_slab, int64_t cand_cap, int n_slabs) {
    const int slab = blockIdx.x * (kChainThreads / 32) + (threadIdx.x >> 5);  // one warp per slab
    if (slab >= n_slabs) return;
    const int2 sb = slab_part[slab];
    if (slab_part[slab + 1].x == sb.x) return;  // no start hit in this slab
    const int base = row_offsets[slab], n = min(row_offsets[slab + 1] - base, 65535);
    const int lane = threadIdx.x & 31;
    const unsigned lt = (1u << lane) - 1u;
    int2 carry = sb;  // (start hits, candidates) before the current 32 input positions
    for (int i0 = 0; i0 < n; i0 += 32) {
        const int i = i0 + lane;  // input position
        int pos = 0;
        uint8_t f = 0;
        if (i < n) {
            pos = hit_pos[base + i];
            f = flags[base + pos];
        }
        const unsigned ms = __ballot_sync(0xffffffffu, f & 1), mc = __ballot_sync(0xffffffffu, f & 2);
        if (f) {
            const int64_t ps = carry.x + __popc(ms & lt);
            if (start_hits && ps < start_cap) start_hits[ps] = base + i;
            if (f & 2) {
                const int64_t c = carry.y + __popc(mc & lt);
                if (c < cand_cap) {
                    cand_start[c] = base + pos;
                    cand_slab[c] = slab;
                }
            }
        }
        carry.x += __popc(ms);
        carry.y += __popc(mc);
    }
}

// Parity/debug export of one link array: sorted space -> input-order positions and values.  dir = +1 / -1 is the
// row offset of the link targets.
// `mutual` != NULL: the link is kept only if mutual[link] points back (the cleaned link computed on the fly, reading S3).
__global__ void __launch_bounds__(kChainThreads)
export_links_kernel(const int32_t* __restrict__ row_offsets, const uint16_t* __restrict__ hit_idx,
                    const int32_t* __restrict__ link, const int32_t* __restrict__ mutual, int dir, int n_slabs,
                    int32_t* __restrict__ out) {
    const int slab = blockIdx.x;
    const int base = row_offsets[slab], n_all = row_offsets[slab + 1] - base;
    const int n = min(n_all, 65535);
    // the target lies in the adjacent row, or two rows away where S2 bridged a missing row (reading A2'); row offsets
    // of a neighbouring instance are never selected because a link stays inside its instance
    const int t1 = min(max(slab + dir, 0), n_slabs - 1), t2 = min(max(slab + 2 * dir, 0), n_slabs - 1);
    const int b1 = row_offsets[t1], b2 = row_offsets[t2], e1 = row_offsets[t1 + 1];
    for (int i = threadIdx.x; i < n; i += kChainThreads) {
        int32_t v = link[base + i];
        if (mutual && v >= 0 && mutual[v] != base + i) v = -1;
        const int tbase = (v >= b1 && v < e1) ? b1 : b2;
        out[base + hit_idx[base + i]] = v < 0 ? -1 : tbase + (int32_t)hit_idx[v];
    }
    for (int i = n + threadIdx.x; i < n_all; i += kChainThreads) out[base + i] = -1;
}

// Two-level scan for long inputs (the per-slab counts: ~570 k entries at 100 windows, where one CTA takes 0.43 ms):
// every CTA scans a tile of 4096 entries in place and reports its total; the tile totals go through the one-CTA scan;
// a last pass adds the tile offsets.
constexpr int kTile = kScanThreads * 4;

__global__ void __launch_bounds__(kScanThreads)
scan_tiles_kernel(int2* __restrict__ part, int64_t m, int2* __restrict__ tile_sums) {
    __shared__ int2 s_warp[kScanThreads / 32];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int64_t i0 = (int64_t)blockIdx.x * kTile + (int64_t)threadIdx.x * 4;
    int2 v[4];
    int2 sum = make_int2(0, 0);
#pragma unroll
    for (int q = 0; q < 4; q++) {
        v[q] = i0 + q < m ? part[i0 + q] : make_int2(0, 0);
        sum.x += v[q].x;
        sum.y += v[q].y;
    }
    int2 incl = sum;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int a = __shfl_up_sync(0xffffffffu, incl.x, d), b = __shfl_up_sync(0xffffffffu, incl.y, d);
        if (lane >= d) { incl.x += a; incl.y += b; }
    }
    if (lane == 31) s_warp[wid] = incl;
    __syncthreads();
    int2 off = make_int2(0, 0), tot = make_int2(0, 0);
#pragma unroll
    for (int k = 0; k < kScanThreads / 32; k++) {
        const int2 w = s_warp[k];
        if (k < wid) { off.x += w.x; off.y += w.y; }
        tot.x += w.x;
        tot.y += w.y;
    }
    int2 run = make_int2(off.x + incl.x - sum.x, off.y + incl.y - sum.y);
#pragma unroll
    for (int q = 0; q < 4; q++) {
        if (i0 + q < m) part[i0 + q] = run;
        run.x += v[q].x;
        run.y += v[q].y;
    }
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(256)
add_tile_offsets_kernel(int2* __restrict__ part, int64_t m, const int2* __restrict__ tile_sums, int n_tiles) {
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i < m) {
        const int2 o = tile_sums[i / kTile];
        int2 v = part[i];
        v.x += o.x;
        v.y += o.y;
        part[i] = v;
    } else if (i == m) {
        part[m] = tile_sums[n_tiles];  // the totals
    }
}

// returns the kernels launched
int launch_scan_int2_long(int2* part, int64_t m, int2* tile_sums, int64_t* counts, int c0, int c1, cudaStream_t s) {
    if (m <= 4 * kTile) {
        scan_int2_kernel<<<1, kScanThreads, 0, s>>>(part, nullptr, 1, 0, m, counts, c0, c1);
        return 1;
    }
    const int n_tiles = div_up(m, kTile);
    scan_tiles_kernel<<<n_tiles, kScanThreads, 0, s>>>(part, m, tile_sums);
    scan_int2_kernel<<<1, kScanThreads, 0, s>>>(tile_sums, nullptr, 1, 0, n_tiles, counts, c0, c1);
    add_tile_offsets_kernel<<<div_up(m + 1, 256), 256, 0, s>>>(part, m, tile_sums, n_tiles);
    return 3;
}

void launch_scan_int2(int2* part, const int64_t* m_dev, int64_t m_div, int64_t m_cap, int64_t m_host, int64_t* counts,
                      int c0, int c1, cudaStream_t s) {
    scan_int2_kernel<<<1, kScanThreads, 0, s>>>(part, m_dev, m_div, m_cap, m_host, counts, c0, c1);
}

int launch_chains(const DevGeom& g, const Workspace& w, const Problem& p, const ChainOut& u, cudaStream_t s) {
    const int slabs = p.n_inst * g.R;
    if (slabs == 0) return 0;
    const int grid = div_up(slabs, kChainThreads / 32);
    clean_flags_kernel<<<grid, kChainThreads, 0, s>>>(g, p.row_offsets, w.up_raw, w.dn_raw, w.up, w.claim, w.flags,
                                                      w.slab_part, slabs);
    const int scans = launch_scan_int2_long(w.slab_part, slabs, w.scan_tmp, w.counts, 0, 1, s);
    chain_write_kernel<<<grid, kChainThreads, 0, s>>>(p.row_offsets, w.hit_pos, w.flags, w.slab_part, u.start_hits,
                                                      u.start_cap, w.cand_start, w.cand_slab, w.Cmax, slabs);
    return 2 + scans;
}

int launch_export_links(const DevGeom& g, const Workspace& w, const Problem& p, const int32_t* link,
                        const int32_t* mutual, int dir, int32_t* out, cudaStream_t s) {
    const int slabs = p.n_inst * g.R;
    if (slabs == 0 || !out) return 0;
    export_links_kernel<<<slabs, kChainThreads, 0, s>>>(p.row_offsets, w.hit_idx, link, mutual, dir, slabs, out);
    return 1;
}

}  // namespace tpc
