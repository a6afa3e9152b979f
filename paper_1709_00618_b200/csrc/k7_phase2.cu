// Phase 2: sector merger + track refit -- "The second phase merges the track segments found in the individual
// sectors to final tracks and performs a track refit" (PAPER.md:33 names a GPU prototype of this fit;
// SURVEY.md 8(f) NEXT-3).  Readings M1-M4 of DESIGN.md "Phase 2".  Works on the workspace of the preceding
// tpc_track_sectors call: a final track's kept hits are the set bits of its kept-row mask (S6 record), each hit is
// tl_rowhit[candidate][row] in the sorted row, so no index is searched.
//
//   refit_tracks   one thread per final track: M1 over its kept hits (seed, one step outward, prior reset, filter
//                  inward); also notes the rows and the outermost hit the matching needs
//   inst_first     first track of every sector instance (tracks are in candidate = instance order): binary search
//   match          one thread per track A that ends before the last pad row: scan the tracks of the two neighbouring
//                  sector instances with an integer pre-filter (first_row in (last_row(A), last_row(A) + 10]), then
//                  rotate + transport the candidate's refitted state to A's outermost row; A keeps its nearest
//                  candidate, every B keeps its nearest A through a 64-bit atomicMin of (d2, A)
//   link           mutual choices become links
//   heads/scan     merged tracks are numbered in ascending innermost segment (deterministic: count, scan, rank)
//   chain_fit      one thread per merged track: single segments copy their refit, chains get ONE filter pass from
//                  the outermost hit of the outermost segment inward, rotating (kf_rotate) at the sector boundaries
#include "kf_math.cuh"

namespace tpc {

constexpr int kP2Threads = 128;
constexpr int kMergeGap = 10;       // reading M3: first_row(B) - last_row(A) <= 10
constexpr float kMergeCut = 2.0f;   // reading M3: |dy|, |dz| <= 2 cm
constexpr unsigned long long kNoPrev = ~0ull;

struct P2Args {
    const int32_t* row_offsets;
    const float2* hit_yz;
    const int32_t* cand_slab;
    const uint16_t* tl_rowhit;
    const uint32_t* tl_sel;
    const int32_t* trk_cand;
    const int64_t* counts;  // phase-1 counts of the workspace: [3] = final tracks
    int64_t Tmax;
    float* p2_par;
    float* p2_cov;
    float* p2_chi2;
    int4* p2_info;
    float2* p2_last;
    int32_t* p2_first;
    int32_t* p2_rowstart;
    int32_t* p2_sorted;
    unsigned long long* p2_best_prev;
    int32_t* p2_best_next;
    int32_t* p2_next;
    int32_t* p2_prev;
    int2* p2_part;
    int2* p2_chain;  // [Tmax / 2 + 1] (innermost segment, merged-track index) of every chain
    int64_t* p2_counts;
    int32_t n_inst;
};

// The kept hits of one final track, walked from the outermost row inward.
struct HitWalk {
    const uint32_t* mask;    // kept-row mask words of the S6 record
    const uint16_t* rowhit;  // tl_rowhit of the candidate
    const int32_t* ro;       // row offsets of the sector instance
    int words;
};

__device__ __forceinline__ HitWalk hit_walk(const DevGeom& g, const P2Args& a, int c) {
    const int inst = a.cand_slab[c] / g.R;
    return HitWalk{a.tl_sel + (size_t)c * g.sel_stride, a.tl_rowhit + (size_t)c * g.RP,
                   a.row_offsets + (size_t)inst * g.R, g.sel_words};
}

__device__ __forceinline__ float2 hit_at(const P2Args& a, const HitWalk& h, int row) {
    return a.hit_yz[h.ro[row] + (int)h.rowhit[row]];
}

// rows of the first, the (n/2)-th (ascending, 0-based) and the last kept hit; returns n
__device__ __forceinline__ int kept_rows(const HitWalk& h, int& r_first, int& r_mid, int& r_last) {
    int n = 0;
    for (int q = 0; q < h.words; q++) n += __popc(h.mask[q]);
    r_first = r_mid = r_last = 0;
    int seen = 0;
    bool have_first = false;
    const int want = n >> 1;
    for (int q = 0; q < h.words; q++) {
        const uint32_t m = h.mask[q];
        if (!m) continue;
        if (!have_first) { r_first = 32 * q + __ffs(m) - 1; have_first = true; }
        r_last = 32 * q + 31 - __clz(m);
        const int k = __popc(m);
        if (want >= seen && want < seen + k) r_mid = 32 * q + (int)__fns(m, 0, want - seen + 1);
        seen += k;
    }
    return n;
}

// One inward filter pass over a segment's kept hits (reading M1 body).  The state sits at plane x (absolute frame
// reference yref/zref as in S5: st.y, st.z are relative to the last attached hit).  Returns false on a failed
// transport.
__device__ __forceinline__ bool filter_inward(const DevGeom& g, const P2Args& a, const HitWalk& h, KfState& st, float& x,
                                              float& yref, float& zref, float& chi2, int& nhits) {
    for (int q = h.words - 1; q >= 0; q--) {
        uint32_t m = h.mask[q];
        while (m) {
            const int b = 31 - __clz(m);
            m &= ~(1u << b);
            const int row = 32 * q + b;
            const float xr = g.row_x[row];
            const float2 hit = hit_at(a, h, row);
            if (xr != x) {
                if (!kf_transport(st, xr - x, g.cB, g.max_s)) return false;
                x = xr;
            }
            chi2 += kf_update(st, hit.x - yref, hit.y - zref, g.sy2, g.sz2);
            yref = hit.x;
            zref = hit.y;
            nhits++;
        }
    }
    return true;
}

// Seed of a segment (its first / middle / last kept hit), moved in one step to its outermost hit's row, covariance =
// prior (reading M1).  Returns false if the seed or the step fails.
__device__ __forceinline__ bool seed_outer(const DevGeom& g, const P2Args& a, const HitWalk& h, KfState& st, float& x,
                                           float& yref, float& zref, int& r_first, int& r_last, int& n) {
    int r_mid;
    n = kept_rows(h, r_first, r_mid, r_last);
    if (n < 3) return false;
    const float2 h0 = hit_at(a, h, r_first), h1 = hit_at(a, h, r_mid), h2 = hit_at(a, h, r_last);
    const float x0 = g.row_x[r_first], x1 = g.row_x[r_mid], x2 = g.row_x[r_last];
    yref = h0.x;
    zref = h0.y;
    if (!kf_seed(st, x0, 0.0f, 0.0f, x1, h1.x - yref, x2, h2.x - yref, h2.y - zref, g.cB, g.max_s, g.p0)) return false;
    if (!kf_transport(st, x2 - x0, g.cB, g.max_s)) return false;
    x = x2;
    st.c00 = g.p0[0]; st.c11 = g.p0[1]; st.c22 = g.p0[2]; st.c33 = g.p0[3]; st.c44 = g.p0[4];
    st.c10 = st.c20 = st.c21 = st.c30 = st.c31 = st.c32 = st.c40 = st.c41 = st.c42 = st.c43 = 0.0f;
    return true;
}

__device__ __forceinline__ void store_fit(float* par, float* cov, const KfState& st, float yref, float zref, bool ok) {
    par[0] = ok ? st.y + yref : 0.0f;
    par[1] = ok ? st.z + zref : 0.0f;
    par[2] = ok ? st.s : 0.0f;
    par[3] = ok ? st.t : 0.0f;
    par[4] = ok ? st.k : 0.0f;
    const float v[15] = {st.c00, st.c10, st.c11, st.c20, st.c21, st.c22, st.c30, st.c31,
                         st.c32, st.c33, st.c40, st.c41, st.c42, st.c43, st.c44};
#pragma unroll
    for (int q = 0; q < 15; q++) cov[q] = ok ? v[q] : 0.0f;
}

__global__ void __launch_bounds__(kP2Threads)
refit_tracks_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ P2Args a) {
    const int64_t n_trk = min(a.counts[3], a.Tmax);
    for (int64_t t = (int64_t)blockIdx.x * kP2Threads + threadIdx.x; t < n_trk; t += (int64_t)gridDim.x * kP2Threads) {
        const int c = a.trk_cand[t];
        const HitWalk h = hit_walk(g, a, c);
        KfState st = {};
        float x = 0.0f, yref = 0.0f, zref = 0.0f, chi2 = 0.0f;
        int r_first = 0, r_last = 0, n = 0, nhits = 0;
        bool ok = seed_outer(g, a, h, st, x, yref, zref, r_first, r_last, n);
        const float2 last = n > 0 ? hit_at(a, h, r_last) : make_float2(0.0f, 0.0f);
        if (ok) ok = filter_inward(g, a, h, st, x, yref, zref, chi2, nhits);
        store_fit(a.p2_par + t * 5, a.p2_cov + t * 15, st, yref, zref, ok);
        a.p2_chi2[t] = ok ? chi2 : 0.0f;
        a.p2_info[t] = make_int4(ok ? 1 : 0, r_first, r_last, n);
        a.p2_last[t] = last;
        a.p2_best_prev[t] = kNoPrev;
        a.p2_best_next[t] = -1;
        a.p2_next[t] = -1;
        a.p2_prev[t] = -1;
        if (!ok) atomicAdd((unsigned long long*)&a.p2_counts[2], 1ull);
    }
}

__device__ __forceinline__ int track_inst(const DevGeom& g, const P2Args& a, int64_t t) {
    return a.cand_slab[a.trk_cand[t]] / g.R;
}

// p2_first[i] = first track whose sector instance is >= i (tracks are in instance order); entry n_inst = n_tracks
__global__ void __launch_bounds__(kP2Threads)
inst_first_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ P2Args a) {
    const int64_t n_trk = min(a.counts[3], a.Tmax);
    const int i = blockIdx.x * kP2Threads + threadIdx.x;
    if (i > a.n_inst) return;
    int64_t lo = 0, hi = n_trk;  // first t in [0, n_trk] with inst(t) >= i
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (track_inst(g, a, mid) < i) lo = mid + 1; else hi = mid;
    }
    a.p2_first[i] = (int32_t)lo;
}

// Index for the matching: per sector instance the fitted tracks ordered by their first row (counting sort in shared
// memory, one CTA per instance).  A track can only be continued by tracks that begin in the kMergeGap rows after its
// last row, so the matching reads that slice instead of all tracks of the neighbouring sectors.  The order inside a
// row's bucket is not defined; the matching does not depend on it (minimum over (distance, track index)).
__global__ void __launch_bounds__(kP2Threads)
index_tracks_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ P2Args a) {
    __shared__ int s_cnt[kMaxRows + 2];
    const int inst = blockIdx.x;
    const int t0 = a.p2_first[inst], t1 = a.p2_first[inst + 1];
    for (int r = threadIdx.x; r <= g.R; r += kP2Threads) s_cnt[r] = 0;
    __syncthreads();
    for (int t = t0 + threadIdx.x; t < t1; t += kP2Threads) {
        const int4 it = a.p2_info[t];
        if (it.x) atomicAdd(&s_cnt[it.y], 1);
    }
    __syncthreads();
    if (threadIdx.x < 32) {  // exclusive scan of the R counts by one warp; s_cnt[r] becomes the bucket's start
        int carry = 0;
        for (int r0 = 0; r0 <= g.R; r0 += 32) {
            const int r = r0 + threadIdx.x;
            const int v = r < g.R ? s_cnt[r] : 0;
            int x = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, x, d);
                if ((int)threadIdx.x >= d) x += y;
            }
            if (r <= g.R) {
                s_cnt[r] = carry + x - v;
                a.p2_rowstart[(size_t)inst * (g.R + 1) + r] = t0 + carry + x - v;
            }
            carry += __shfl_sync(0xffffffffu, x, 31);
        }
    }
    __syncthreads();
    for (int t = t0 + threadIdx.x; t < t1; t += kP2Threads) {
        const int4 it = a.p2_info[t];
        if (it.x) a.p2_sorted[t0 + atomicAdd(&s_cnt[it.y], 1)] = t;
    }
}

// One WARP per track A (grid-stride): the lanes read the tracks of a neighbouring sector instance that begin in the
// kMergeGap rows after A's last row (index_tracks_kernel), 32 at a time, and those pay for the extrapolation.
__global__ void __launch_bounds__(kP2Threads)
match_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ P2Args a) {
    const int64_t n_trk = min(a.counts[3], a.Tmax);
    const int lane = threadIdx.x & 31;
    const int64_t n_warps = (int64_t)gridDim.x * (kP2Threads / 32);
    for (int64_t ta = (int64_t)blockIdx.x * (kP2Threads / 32) + (threadIdx.x >> 5); ta < n_trk; ta += n_warps) {
        const int4 ia = a.p2_info[ta];
        const int la = ia.z;
        if (ia.w < 1 || la >= g.R - 1) continue;  // reaches the last pad row: nothing can continue it (warp-uniform)
        const int inst = track_inst(g, a, ta);
        const int window = (inst + g.inst_phase) / g.spe, sec = (inst + g.inst_phase) % g.spe;
        const int side = sec >= g.spe_half ? 1 : 0, phi = sec % g.spe_half;
        const float2 ha = a.p2_last[ta];
        const float xa = g.row_x[la];
        const int row_hi = min(la + kMergeGap, g.R - 1);  // last row a continuation may begin in
        float best_d2 = __int_as_float(0x7f800000);
        int best_b = 0x7fffffff;
        // the two neighbouring sectors of the same side and window.  Rotation from B's frame into A's: by -2h when B
        // is the next sector in azimuth (dir = +1), by +2h when it is the previous one.
        for (int dir = -1; dir <= 1; dir += 2) {
            const int phi_b = (phi + dir + g.spe_half) % g.spe_half;
            const int inst_b = window * g.spe + side * g.spe_half + phi_b - g.inst_phase;
            if (inst_b < 0 || inst_b >= a.n_inst) continue;  // the neighbour is not part of this call (chunked jobs)
            const float sa = dir > 0 ? -g.sin_2h : g.sin_2h;
            const int32_t* rs = a.p2_rowstart + (size_t)inst_b * (g.R + 1);
            const int k_end = rs[row_hi + 1];
            for (int k = rs[la + 1] + lane; k < k_end; k += 32) {
                const int tb = a.p2_sorted[k];
                const int4 ib = a.p2_info[tb];
                if (!(ib.x && ib.y > la && ib.y - la <= kMergeGap)) continue;  // holds by construction of the slice
                KfState st;
                const float* p = a.p2_par + (size_t)tb * 5;
                const float* q = a.p2_cov + (size_t)tb * 15;
                st.y = p[0]; st.z = p[1]; st.s = p[2]; st.t = p[3]; st.k = p[4];
                st.c00 = q[0]; st.c10 = q[1]; st.c11 = q[2]; st.c20 = q[3]; st.c21 = q[4]; st.c22 = q[5];
                st.c30 = q[6]; st.c31 = q[7]; st.c32 = q[8]; st.c33 = q[9]; st.c40 = q[10]; st.c41 = q[11];
                st.c42 = q[12]; st.c43 = q[13]; st.c44 = q[14];
                float xr;
                if (!kf_rotate(st, st.y, g.row_x[ib.y], g.cos_2h, sa, g.cB, g.max_s, xr)) continue;
                if (!kf_transport(st, xa - xr, g.cB, g.max_s)) continue;
                const float dy = st.y - ha.x, dz = st.z - ha.y;
                if (!(fabsf(dy) <= kMergeCut && fabsf(dz) <= kMergeCut)) continue;
                const float d2 = dy * dy + dz * dz;
                if (d2 < best_d2 || (d2 == best_d2 && tb < best_b)) { best_d2 = d2; best_b = tb; }
                atomicMin(&a.p2_best_prev[tb], ((unsigned long long)__float_as_uint(d2) << 32) | (unsigned long long)ta);
            }
        }
        // nearest over the lanes; an exact tie of d2 goes to the lower track index
        unsigned long long key = ((unsigned long long)__float_as_uint(best_d2) << 32) | (unsigned)best_b;
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) {
            const unsigned long long other = __shfl_xor_sync(0xffffffffu, key, o);
            key = other < key ? other : key;
        }
        if (lane == 0)
            a.p2_best_next[ta] = (unsigned)(key & 0xffffffffull) == 0x7fffffffu ? -1 : (int)(key & 0xffffffffull);
    }
}

__global__ void __launch_bounds__(kP2Threads)
link_kernel(const __grid_constant__ P2Args a) {
    const int64_t n_trk = min(a.counts[3], a.Tmax);
    const int64_t ta = (int64_t)blockIdx.x * kP2Threads + threadIdx.x;
    if (ta >= n_trk) return;
    const int tb = a.p2_best_next[ta];
    if (tb >= 0 && (int64_t)(a.p2_best_prev[tb] & 0xffffffffull) == ta) {
        a.p2_next[ta] = tb;
        a.p2_prev[tb] = (int32_t)ta;
        atomicAdd((unsigned long long*)&a.p2_counts[1], 1ull);
    }
}

// heads (tracks without a predecessor) and chain heads (heads with a successor) per block of 256 tracks
__global__ void __launch_bounds__(256)
heads_kernel(const __grid_constant__ P2Args a) {
    __shared__ int s_cnt[2];
    const int64_t n_trk = min(a.counts[3], a.Tmax);
    for (int64_t blk = blockIdx.x; blk * 256 < n_trk; blk += gridDim.x) {
        if (threadIdx.x < 2) s_cnt[threadIdx.x] = 0;
        __syncthreads();
        const int64_t t = blk * 256 + threadIdx.x;
        const int head = (t < n_trk && a.p2_prev[t] < 0) ? 1 : 0;
        const int chain = (head && a.p2_next[t] >= 0) ? 1 : 0;
        const int n = __reduce_add_sync(0xffffffffu, head), nc = __reduce_add_sync(0xffffffffu, chain);
        if ((threadIdx.x & 31) == 0) {
            if (n) atomicAdd(&s_cnt[0], n);
            if (nc) atomicAdd(&s_cnt[1], nc);
        }
        __syncthreads();
        if (threadIdx.x == 0) a.p2_part[blk] = make_int2(s_cnt[0], s_cnt[1]);
        __syncthreads();
    }
}

// Per-track outputs, the merged-track records of single segments, and the list of chains (merged tracks of two or
// more segments) for chain_fit_kernel; merged tracks are numbered in ascending innermost segment.
__global__ void __launch_bounds__(256)
merged_out_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ P2Args a, const Phase2Out o) {
    __shared__ int2 s_warp[8];
    const int64_t n_trk = min(a.counts[3], a.Tmax);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int64_t blk = blockIdx.x; blk * 256 < n_trk; blk += gridDim.x) {
        const int64_t t = blk * 256 + threadIdx.x;
        const bool head = t < n_trk && a.p2_prev[t] < 0;
        const bool chain = head && a.p2_next[t] >= 0;
        const unsigned hm = __ballot_sync(0xffffffffu, head), cm = __ballot_sync(0xffffffffu, chain);
        if (lane == 0) s_warp[wid] = make_int2(__popc(hm), __popc(cm));
        __syncthreads();
        const int2 part = a.p2_part[blk];
        int64_t m = part.x + __popc(hm & ((1u << lane) - 1u));
        int64_t e = part.y + __popc(cm & ((1u << lane) - 1u));
        for (int k = 0; k < wid; k++) { m += s_warp[k].x; e += s_warp[k].y; }
        __syncthreads();
        if (t < n_trk) {  // per-track outputs
            if (o.seg_next) o.seg_next[t] = a.p2_next[t];
            if (o.seg_prev) o.seg_prev[t] = a.p2_prev[t];
            if (o.seg_ok) o.seg_ok[t] = a.p2_info[t].x;
            if (o.seg_chi2) o.seg_chi2[t] = a.p2_chi2[t];
            if (o.seg_params)
#pragma unroll
                for (int q = 0; q < 5; q++) o.seg_params[t * 5 + q] = a.p2_par[t * 5 + q];
            if (o.seg_cov)
#pragma unroll
                for (int q = 0; q < 15; q++) o.seg_cov[t * 15 + q] = a.p2_cov[t * 15 + q];
        }
        if (!head) continue;
        // every chain goes on the list, also one whose merged index lies beyond the caller's capacity: chain_fit_kernel
        // walks all p2_counts[4] entries and skips those itself (an unwritten entry would be stale workspace memory)
        if (chain) a.p2_chain[e] = make_int2((int)t, (int)m);
        if (m >= o.mtrk_capacity) continue;
        if (o.mtrk_first) o.mtrk_first[m] = (int32_t)t;
        if (chain) continue;  // fitted by chain_fit_kernel, one dense thread per chain
        // not merged: the refit of the track alone
        const int4 info = a.p2_info[t];
        if (o.mtrk_nseg) o.mtrk_nseg[m] = 1;
        if (o.mtrk_nhits) o.mtrk_nhits[m] = info.x ? info.w : 0;
        if (o.mtrk_ok) o.mtrk_ok[m] = info.x;
        if (o.mtrk_chi2) o.mtrk_chi2[m] = a.p2_chi2[t];
        if (o.mtrk_params)
#pragma unroll
            for (int q = 0; q < 5; q++) o.mtrk_params[m * 5 + q] = a.p2_par[t * 5 + q];
        if (o.mtrk_cov)
#pragma unroll
            for (int q = 0; q < 15; q++) o.mtrk_cov[m * 15 + q] = a.p2_cov[t * 15 + q];
        if (!info.x) atomicAdd((unsigned long long*)&a.p2_counts[3], 1ull);
    }
}

// Reading M4: one thread per chain; seed on the outermost segment, filter inward through the chain, rotating the
// state and covariance at every sector boundary.
__global__ void __launch_bounds__(kP2Threads)
chain_fit_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ P2Args a, const Phase2Out o) {
    const int64_t n_chain = a.p2_counts[4];
    for (int64_t e = (int64_t)blockIdx.x * kP2Threads + threadIdx.x; e < n_chain; e += (int64_t)gridDim.x * kP2Threads) {
        const int2 ent = a.p2_chain[e];
        const int64_t t = ent.x, m = ent.y;
        if (m >= o.mtrk_capacity) continue;
        int nseg = 1;
        int64_t tail = t;
        while (a.p2_next[tail] >= 0 && nseg < 64) { tail = a.p2_next[tail]; nseg++; }
        KfState st = {};
        float x = 0.0f, yref = 0.0f, zref = 0.0f, chi2 = 0.0f;
        int nhits = 0;
        int64_t cur = tail;
        HitWalk h = hit_walk(g, a, a.trk_cand[cur]);
        // The outermost segment is not fitted again: refit_tracks_kernel has just run exactly this seed + inward pass
        // over its kept hits (reading M1 = the first leg of M4) and left the state at its innermost kept hit in
        // p2_par / p2_cov / p2_chi2.  The state is taken back into the frame relative to that hit; what is lost is
        // the rounding of y and z to fp32 when they were stored (<= 4e-6 cm at y ~ 100 cm).
        const int4 tinfo = a.p2_info[tail];
        bool ok = tinfo.x != 0;
        if (ok) {
            const float2 h0 = hit_at(a, h, tinfo.y);
            const float* sp = a.p2_par + tail * 5;
            const float* sc = a.p2_cov + tail * 15;
            yref = h0.x;
            zref = h0.y;
            st.y = sp[0] - yref; st.z = sp[1] - zref; st.s = sp[2]; st.t = sp[3]; st.k = sp[4];
            st.c00 = sc[0]; st.c10 = sc[1]; st.c11 = sc[2]; st.c20 = sc[3]; st.c21 = sc[4]; st.c22 = sc[5];
            st.c30 = sc[6]; st.c31 = sc[7]; st.c32 = sc[8]; st.c33 = sc[9]; st.c40 = sc[10]; st.c41 = sc[11];
            st.c42 = sc[12]; st.c43 = sc[13]; st.c44 = sc[14];
            x = g.row_x[tinfo.y];
            chi2 = a.p2_chi2[tail];
            nhits = tinfo.w;
        }
        while (ok && cur != t) {
            const int64_t inner = a.p2_prev[cur];
            const int sec_o = (track_inst(g, a, cur) + g.inst_phase) % g.spe_half;  // azimuth index (same side)
            const int sec_i = (track_inst(g, a, inner) + g.inst_phase) % g.spe_half;
            // rotation from the outer segment's frame into the inner one's: +2h when the inner sector is the next in
            // azimuth, -2h when it is the previous one
            const bool inner_is_next = ((sec_o + 1) % g.spe_half) == sec_i;
            float xr;
            ok = kf_rotate(st, st.y + yref, x, g.cos_2h, inner_is_next ? g.sin_2h : -g.sin_2h, g.cB, g.max_s, xr);
            x = xr;
            yref = 0.0f;  // kf_rotate leaves the absolute y in st.y
            cur = inner;
            if (ok) {
                h = hit_walk(g, a, a.trk_cand[cur]);
                ok = filter_inward(g, a, h, st, x, yref, zref, chi2, nhits);
            }
        }
        if (o.mtrk_nseg) o.mtrk_nseg[m] = nseg;
        if (o.mtrk_nhits) o.mtrk_nhits[m] = ok ? nhits : 0;
        if (o.mtrk_ok) o.mtrk_ok[m] = ok ? 1 : 0;
        if (o.mtrk_chi2) o.mtrk_chi2[m] = ok ? chi2 : 0.0f;
        float par[5], cov[15];
        store_fit(par, cov, st, yref, zref, ok);
        if (o.mtrk_params)
#pragma unroll
            for (int q = 0; q < 5; q++) o.mtrk_params[m * 5 + q] = par[q];
        if (o.mtrk_cov)
#pragma unroll
            for (int q = 0; q < 15; q++) o.mtrk_cov[m * 15 + q] = cov[q];
        if (!ok) atomicAdd((unsigned long long*)&a.p2_counts[3], 1ull);
    }
}

__global__ void p2_counts_kernel(const int64_t* __restrict__ c, int64_t* __restrict__ user) {
    if (threadIdx.x < 4) user[threadIdx.x] = c[threadIdx.x];
}

// defined in k34_links_chains.cu
void launch_scan_int2(int2* part, const int64_t* m_dev, int64_t m_div, int64_t m_cap, int64_t m_host, int64_t* counts,
                      int c0, int c1, cudaStream_t s);

int launch_phase2(const DevGeom& g, const Workspace& w, const Problem& p, const Phase2Out& o, cudaStream_t s) {
    cudaMemsetAsync(w.p2_counts, 0, sizeof(int64_t) * 8, s);
    int launches = 0;
    if (p.n_clusters > 0) {
        const P2Args a{p.row_offsets, w.hit_yz,     w.cand_slab,    w.tl_rowhit,    w.tl_sel,  w.trk_cand, w.counts,
                       w.Tmax,        w.p2_par,     w.p2_cov,       w.p2_chi2,      w.p2_info, w.p2_last,  w.p2_first,
                       w.p2_rowstart, w.p2_sorted, w.p2_best_prev, w.p2_best_next, w.p2_next,   w.p2_prev,      w.p2_part, w.p2_chain, w.p2_counts, p.n_inst};
        // the track count lives on the device: grids are sized by its bound and bounded by it inside
        const int64_t tb = div_up(w.Tmax, kP2Threads);
        const int grid_t = (int)(tb < 148 * 64 ? tb : 148 * 64);
        refit_tracks_kernel<<<grid_t, kP2Threads, 0, s>>>(g, a);
        inst_first_kernel<<<div_up((int64_t)p.n_inst + 1, kP2Threads), kP2Threads, 0, s>>>(g, a);
        index_tracks_kernel<<<p.n_inst, kP2Threads, 0, s>>>(g, a);
        const int64_t mb = div_up(w.Tmax, kP2Threads / 32);
        match_kernel<<<(int)(mb < 148 * 16 ? mb : 148 * 16), kP2Threads, 0, s>>>(g, a);
        link_kernel<<<(unsigned)tb, kP2Threads, 0, s>>>(a);
        const int64_t hb = div_up(w.Tmax, 256);
        const int grid_h = (int)(hb < 148 * 16 ? hb : 148 * 16);
        heads_kernel<<<grid_h, 256, 0, s>>>(a);
        launch_scan_int2(w.p2_part, w.counts + 3, 256, w.Tmax, 0, w.p2_counts, 0, 4, s);  // [0] heads, [4] chains
        merged_out_kernel<<<grid_h, 256, 0, s>>>(g, a, o);
        const int64_t cb = div_up(w.Tmax / 2 + 1, kP2Threads);
        chain_fit_kernel<<<(int)(cb < 148 * 64 ? cb : 148 * 64), kP2Threads, 0, s>>>(g, a, o);
        launches += 9;
    }
    p2_counts_kernel<<<1, 32, 0, s>>>(w.p2_counts, o.counts2);
    return launches + 1;
}

}  // namespace tpc
