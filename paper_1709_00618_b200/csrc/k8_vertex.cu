// Time-coordinate tracking: vertex estimate -- "the tracking will run in time coordinate first to estimate the vertex
// and only then convert to spacial coordinates" (continuous read-out).
// Readings T1-T3 of DESIGN.md.  Works on the merged tracks of the preceding tpc_merge_refit call.
//
//   track_vertex   one thread per merged track: closest approach to the beam line (closed form), histogram vote
//   vertex_seeds   one CTA per event window: 3-bin sums of its histogram in shared memory, local maxima, seeds
//                  compacted in ascending bin
//   vertex_scan    vertex numbering = exclusive scan of the seeds per window (one CTA)
//   vertex_sums    one thread per merged track: integer (fixed-point) atomics of z_v into the seeds within 1.5 cm, so
//                  that the mean does not depend on the order of the atomics
//   vertex_assign  one thread per merged track: nearest vertex of its window within 3 cm; vertex positions and counts
#include "tpc_common.cuh"

namespace tpc {

constexpr int kVtxThreads = 256;
constexpr int kVtxMax = 64;          // TPC_VTX_MAX_PER_WINDOW
constexpr float kVtxBin = 0.5f;      // reading T2
constexpr int kVtxMinHits = 30;
constexpr float kVtxMaxDca = 3.0f;
constexpr int kVtxMinSum = 10;
constexpr int kVtxRange = 4;
constexpr float kVtxMeanWin = 1.5f;
constexpr float kVtxAssign = 3.0f;
constexpr float kVtxFixed = 65536.0f;  // fixed-point scale of the z_v sums (fp32 values below 1024 cm are exact)

struct VtxArgs {
    const int32_t* cand_slab;
    const int32_t* trk_cand;
    const int4* p2_info;
    int32_t* hist;
    int32_t* seed;
    int32_t* nseed;
    long long* sum;
    int32_t* cnt;
    uint8_t* like;
    int64_t* counts;
    int32_t n_win;
    int32_t win0;  // window of instance 0 of the call
};

__device__ __forceinline__ int track_window(const DevGeom& g, const VtxArgs& a, int first_seg) {
    const int inst = a.cand_slab[a.trk_cand[first_seg]] / g.R;
    return (inst + g.inst_phase) / g.spe - a.win0;
}

__global__ void __launch_bounds__(kVtxThreads)
track_vertex_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ VtxArgs a, const Phase2Out m,
                    const VertexOut o) {
    const int64_t n_m = min(m.counts2[0], m.mtrk_capacity);
    const int64_t i = (int64_t)blockIdx.x * kVtxThreads + threadIdx.x;
    if (i >= n_m) return;
    float zv = 0.0f, dca = 0.0f;
    uint8_t like = 0;
    if (m.mtrk_ok[i]) {
        const float* p = m.mtrk_params + i * 5;
        const int first = m.mtrk_first[i];
        const float x = g.row_x[a.p2_info[first].y];
        // T1: u, v = position along / across the direction; ds = atan2(-kappa u, 1 + kappa v) / kappa
        const float s = p[2], c = sqrtf((1.0f - s) * (1.0f + s)), kap = g.cB * p[4];
        const float u = x * c + p[0] * s, v = -x * s + p[0] * c;
        const float aa = -kap * u, bb = 1.0f + kap * v;
        float ds;
        if (fabsf(kap) * (fabsf(u) + fabsf(v)) < 1e-5f) {
            ds = -u / bb;
            dca = v;
        } else {
            ds = atan2f(aa, bb) / kap;
            // (sqrt(a^2 + b^2) - 1) / kappa without the cancellation: a^2 + b^2 - 1 = kappa (kappa (u^2 + v^2) + 2 v)
            const float r = sqrtf(aa * aa + bb * bb);
            dca = (kap * (u * u + v * v) + 2.0f * v) / (r + 1.0f);
        }
        zv = fmaf(p[3], ds, p[1]);
        like = 2;
        if (m.mtrk_nhits[i] >= kVtxMinHits && fabsf(dca) <= kVtxMaxDca) {
            like = 3;
            const int b = __float2int_rd((zv + g.vtx_h) / kVtxBin);
            const int w = track_window(g, a, first);
            if (b >= 0 && b < g.vtx_nb && w >= 0 && w < a.n_win) atomicAdd(&a.hist[(size_t)w * g.vtx_nb + b], 1);
        }
    }
    if (o.trk_zv) o.trk_zv[i] = zv;
    if (o.trk_dca) o.trk_dca[i] = dca;
    a.like[i] = like;
}

__global__ void __launch_bounds__(kVtxThreads)
vertex_seeds_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ VtxArgs a) {
    extern __shared__ int32_t s_sum3[];  // [vtx_nb] 3-bin sums
    __shared__ int s_warp[kVtxThreads / 32];
    __shared__ int s_base;
    const int w = blockIdx.x;
    const int nb = g.vtx_nb;
    const int32_t* h = a.hist + (size_t)w * nb;
    for (int b = threadIdx.x; b < nb; b += kVtxThreads)
        s_sum3[b] = h[b] + (b > 0 ? h[b - 1] : 0) + (b + 1 < nb ? h[b + 1] : 0);
    if (threadIdx.x == 0) s_base = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int b0 = 0; b0 < nb; b0 += kVtxThreads) {  // ascending bins; ordered compaction by ballot + warp totals
        const int b = b0 + threadIdx.x;
        bool seed = false;
        if (b < nb) {
            const int s3 = s_sum3[b];
            if (s3 >= kVtxMinSum) {
                seed = true;
                for (int q = b - kVtxRange; q <= b + kVtxRange; q++) {
                    if (q == b || q < 0 || q >= nb) continue;
                    const int oq = s_sum3[q];
                    if (oq > s3 || (oq == s3 && q < b)) seed = false;
                }
            }
        }
        const unsigned mk = __ballot_sync(0xffffffffu, seed);
        if (lane == 0) s_warp[wid] = __popc(mk);
        __syncthreads();
        int pos = s_base + __popc(mk & ((1u << lane) - 1u));
        int tot = 0;
        for (int k = 0; k < kVtxThreads / 32; k++) {
            if (k < wid) pos += s_warp[k];
            tot += s_warp[k];
        }
        if (seed && pos < kVtxMax) a.seed[(size_t)w * kVtxMax + pos] = b;
        __syncthreads();
        if (threadIdx.x == 0) s_base += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) a.nseed[w] = min(s_base, kVtxMax);
}

// exclusive scan of the seeds per window (n_win is a few thousand at most): one CTA, serial over chunks of 256
__global__ void __launch_bounds__(kVtxThreads)
vertex_scan_kernel(const __grid_constant__ VtxArgs a) {
    __shared__ int s_part[kVtxThreads];
    const int per = (a.n_win + kVtxThreads - 1) / kVtxThreads;
    const int lo = min(threadIdx.x * per, a.n_win), hi = min(lo + per, a.n_win);
    int sum = 0;
    for (int w = lo; w < hi; w++) sum += a.nseed[w];
    s_part[threadIdx.x] = sum;
    __syncthreads();
    int off = 0;
    for (int k = 0; k < (int)threadIdx.x; k++) off += s_part[k];
    for (int w = lo; w < hi; w++) {
        const int c = a.nseed[w];
        a.nseed[w] = off;
        off += c;
    }
    if (threadIdx.x == kVtxThreads - 1) {
        a.nseed[a.n_win] = off;
        a.counts[0] = off;
    }
}

__device__ __forceinline__ int n_seeds_of(const VtxArgs& a, int w) { return a.nseed[w + 1] - a.nseed[w]; }

__global__ void __launch_bounds__(kVtxThreads)
vertex_sums_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ VtxArgs a, const Phase2Out m,
                   const VertexOut o) {
    const int64_t n_m = min(m.counts2[0], m.mtrk_capacity);
    const int64_t i = (int64_t)blockIdx.x * kVtxThreads + threadIdx.x;
    if (i >= n_m || a.like[i] != 3) return;
    const int w = track_window(g, a, m.mtrk_first[i]);
    if (w < 0 || w >= a.n_win) return;
    const float zv = o.trk_zv[i];
    const int ns = n_seeds_of(a, w);
    for (int k = 0; k < ns; k++) {
        const float zc = -g.vtx_h + ((float)a.seed[(size_t)w * kVtxMax + k] + 0.5f) * kVtxBin;
        if (fabsf(zv - zc) <= kVtxMeanWin) {
            atomicAdd((unsigned long long*)&a.sum[(size_t)w * kVtxMax + k], (unsigned long long)__float2ll_rn(zv * kVtxFixed));
            atomicAdd(&a.cnt[(size_t)w * kVtxMax + k], 1);
        }
    }
}

__device__ __forceinline__ float vertex_z(const VtxArgs& a, int w, int k) {
    const size_t e = (size_t)w * kVtxMax + k;
    return (float)((double)a.sum[e] / (double)kVtxFixed / (double)max(a.cnt[e], 1));
}

__global__ void __launch_bounds__(kVtxThreads)
vertex_assign_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ VtxArgs a, const Phase2Out m,
                     const VertexOut o) {
    const int64_t n_m = min(m.counts2[0], m.mtrk_capacity);
    const int64_t i = (int64_t)blockIdx.x * kVtxThreads + threadIdx.x;
    // vertex records: the first threads of the grid write them (n_vertices <= n_win * 64)
    const int64_t nv = a.nseed[a.n_win];
    if (i < nv && i < o.vtx_capacity) {
        int lo = 0, hi = a.n_win;  // window of vertex i: last w with nseed[w] <= i
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (a.nseed[mid] <= i) lo = mid; else hi = mid;
        }
        if (o.vtx_z) o.vtx_z[i] = vertex_z(a, lo, (int)(i - a.nseed[lo]));
        if (o.vtx_window) o.vtx_window[i] = lo + a.win0;
    }
    if (i >= n_m) return;
    int best = -1;
    if (a.like[i] >= 2) {
        const int w = track_window(g, a, m.mtrk_first[i]);
        if (w >= 0 && w < a.n_win) {
            const float zv = o.trk_zv[i];
            const int ns = n_seeds_of(a, w);
            float bd = 0.0f;
            for (int k = 0; k < ns; k++) {
                const float d = fabsf(zv - vertex_z(a, w, k));
                if (d <= kVtxAssign && (best < 0 || d < bd)) { best = a.nseed[w] + k; bd = d; }
            }
        }
    }
    if (best >= o.vtx_capacity) best = -1;
    if (o.trk_vtx) o.trk_vtx[i] = best;
    if (best >= 0) {
        if (o.vtx_ntracks) atomicAdd(&o.vtx_ntracks[best], 1);
        atomicAdd((unsigned long long*)&a.counts[1], 1ull);
    }
}

__global__ void vtx_counts_kernel(const int64_t* __restrict__ c, int64_t* __restrict__ user) {
    if (threadIdx.x < 2) user[threadIdx.x] = c[threadIdx.x];
}

int launch_vertices(const DevGeom& g, const Workspace& w, const Problem& p, const Phase2Out& m, const VertexOut& o,
                    cudaStream_t s) {
    const int n_win = w.n_win;
    cudaMemsetAsync(w.vz_counts, 0, sizeof(int64_t) * 2, s);
    cudaMemsetAsync(w.vz_hist, 0, sizeof(int32_t) * (size_t)n_win * g.vtx_nb, s);
    cudaMemsetAsync(w.vz_sum, 0, sizeof(long long) * (size_t)n_win * kVtxMax, s);
    cudaMemsetAsync(w.vz_cnt, 0, sizeof(int32_t) * (size_t)n_win * kVtxMax, s);
    if (o.vtx_ntracks && o.vtx_capacity > 0) cudaMemsetAsync(o.vtx_ntracks, 0, sizeof(int32_t) * o.vtx_capacity, s);
    int launches = 0;
    const int64_t n_m_max = m.mtrk_capacity < w.Tmax ? m.mtrk_capacity : w.Tmax;
    if (p.n_clusters > 0 && o.trk_zv && n_m_max > 0) {  // no merged-track slot: no launch (counts3 = 0, 0)
        const VtxArgs a{w.cand_slab, w.trk_cand, w.p2_info, w.vz_hist, w.vz_seed, w.vz_nseed, w.vz_sum, w.vz_cnt,
                        w.vz_like,   w.vz_counts, n_win,    g.inst_phase / g.spe};
        const int grid_m = div_up(n_m_max, kVtxThreads);
        track_vertex_kernel<<<grid_m, kVtxThreads, 0, s>>>(g, a, m, o);
        const size_t seed_smem = sizeof(int32_t) * (size_t)g.vtx_nb;  // <= kVtxMaxSmemBytes (checked by the caller)
        if (seed_smem > 48 * 1024)  // |z| range beyond ~3 km: opt in (cheap, per call: the size depends on the geometry)
            cudaFuncSetAttribute(vertex_seeds_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)seed_smem);
        vertex_seeds_kernel<<<n_win, kVtxThreads, seed_smem, s>>>(g, a);
        vertex_scan_kernel<<<1, kVtxThreads, 0, s>>>(a);
        vertex_sums_kernel<<<grid_m, kVtxThreads, 0, s>>>(g, a, m, o);
        const int64_t nv_max = (int64_t)n_win * kVtxMax;
        const int64_t need = n_m_max > nv_max ? n_m_max : nv_max;
        vertex_assign_kernel<<<div_up(need, kVtxThreads), kVtxThreads, 0, s>>>(g, a, m, o);
        launches += 5;
    }
    vtx_counts_kernel<<<1, 32, 0, s>>>(w.vz_counts, o.counts3);
    return launches + 1;
}

}  // namespace tpc
