// S5: track following -- "fits track parameters to the track candidate and extrapolates the trajectory through the
// TPC sector volume to pick up additional clusters and refine the fit using a simplified Kalman filter"
// (Fig. 1c); constant Bz only.  Control flow: DESIGN.md "S5" (seed, phase A upward,
// one-step back transport, phase B downward).  One thread per candidate, all arithmetic fp32 in registers.
#include "kf_math.cuh"

namespace tpc {

constexpr int kFollowThreads = 128;

struct FollowCtx {
    const float2* hit_yz;
    const uint16_t* hit_idx;
    const uint16_t* bin_start;
    const int32_t* ro;   // row offsets of this candidate's instance [R+1]
    int slab_base;       // instance * R
    float z0;
    const float* s_rowx; // shared [R]
    float yref, zref;    // the filter state holds (y - yref, z - zref): see follow_kernel
};

struct WorkCount {  // per-thread work counters (roofline arithmetic): summed into counts[6..9] at kernel end
    unsigned transports, updates, examined, searches;
};

// Nearest cluster of the row inside the gate around the predicted (y,z); ties -> lowest local index.
// Returns the sorted position (relative to the row start) or -1; (ym, zm) get its coordinates.
__device__ __forceinline__ int pick_up(const DevGeom& g, const FollowCtx& cx, int r, float yp, float zp, float wy,
                                       float wz, float& ym, float& zm, WorkCount& wc) {
    const int base = cx.ro[r];
    const uint16_t* tbl = cx.bin_start + (size_t)(cx.slab_base + r) * g.nzp;
    const float m = 1e-3f;  // bin margin: the visited bins are a superset of the rounded fp32 window test below
    const int b0 = zbin(zp - wz - m, cx.z0, g.inv_cz, g.nz), b1 = zbin(zp + wz + m, cx.z0, g.inv_cz, g.nz);
    const int j0 = tbl[b0], j1 = tbl[b1 + 1];
    wc.searches++;
    wc.examined += j1 - j0;
    int best = -1, best_idx = 0;
    float bd2 = 0.0f;
    const float2* yz = cx.hit_yz + base;
    for (int j = j0; j < j1; j++) {
        const float2 h = yz[j];
        const float dy = __fsub_rn(h.x, yp), dz = __fsub_rn(h.y, zp);
        if (!(fabsf(dy) <= wy && fabsf(dz) <= wz)) continue;
        const float d2 = __fadd_rn(__fmul_rn(dy, dy), __fmul_rn(dz, dz));
        bool better = best < 0 || d2 < bd2;
        int idx = -1;
        if (!better && d2 == bd2) {
            idx = cx.hit_idx[base + j];
            if (best_idx < 0) best_idx = cx.hit_idx[base + best];
            better = idx < best_idx;
        }
        if (better) {
            best = j;
            best_idx = idx;  // -1 = not loaded yet
            bd2 = d2;
            ym = h.x;
            zm = h.y;
        }
    }
    return best;
}

// One direction of the pick-up loop.  Returns the last visited row.
template <int STEP>
__device__ __forceinline__ int follow_dir(const DevGeom& g, const FollowCtx& cx, KfState& st, int r, float& chi2,
                                          int& nhits, int& last_hit_row, uint16_t* __restrict__ rowhit,
                                          KfState* at_hit, WorkCount& wc) {
    int gap = 0;
    for (;;) {
        const int rn = r + STEP;
        if (rn < 0 || rn >= g.R) break;
        const float xr = cx.s_rowx[rn];
        if (!kf_transport(st, xr - cx.s_rowx[r], g.cB, g.max_s)) break;
        wc.transports++;
        r = rn;
        const float yp = st.y + cx.yref, zp = st.z + cx.zref;
        if (fabsf(yp) > fmaf(xr, g.tan_half, g.edge_margin)) break;
        const float wy = fminf(g.wmax, g.gate * sqrtf(st.c00 + g.sy2));
        const float wz = fminf(g.wmax, g.gate * sqrtf(st.c11 + g.sz2));
        float ym, zm;
        const int j = pick_up(g, cx, r, yp, zp, wy, wz, ym, zm, wc);
        if (j >= 0) {
            rowhit[r] = cx.hit_idx[cx.ro[r] + j];
            chi2 += kf_update(st, ym - cx.yref, zm - cx.zref, g.sy2, g.sz2);
            wc.updates++;
            nhits++;
            gap = 0;
            last_hit_row = r;
            if (at_hit) *at_hit = st;
        } else {
            rowhit[r] = kNoHit;
            if (++gap > g.max_gap) break;
        }
    }
    return r;
}

__global__ void __launch_bounds__(kFollowThreads)
follow_kernel(const __grid_constant__ DevGeom g, const float4* __restrict__ clusters,
              const int32_t* __restrict__ row_offsets, const float2* __restrict__ hit_yz,
              const uint16_t* __restrict__ hit_idx, const uint16_t* __restrict__ bin_start,
              const int32_t* __restrict__ cand_hits, const int32_t* __restrict__ cand_n,
              const int32_t* __restrict__ cand_slab, int64_t* __restrict__ counts, int64_t Cmax,
              float* __restrict__ tl_par, float* __restrict__ tl_cov, float* __restrict__ tl_chi2,
              int32_t* __restrict__ tl_nhits, int32_t* __restrict__ tl_rows, uint16_t* __restrict__ tl_rowhit) {
    __shared__ float s_rowx[kMaxRows + 1];
    for (int i = threadIdx.x; i < g.R; i += kFollowThreads) s_rowx[i] = g.row_x[i];
    __syncthreads();
    const int64_t n_cand = min(counts[1], Cmax);
    const int64_t stride = (int64_t)gridDim.x * kFollowThreads;
    WorkCount wc = {0u, 0u, 0u, 0u};
    for (int64_t c = (int64_t)blockIdx.x * kFollowThreads + threadIdx.x; c < n_cand; c += stride) {
        const int slab0 = cand_slab[c];
        const int inst = slab0 / g.R, r0 = slab0 - inst * g.R;
        const int n = cand_n[c];
        FollowCtx cx;
        cx.hit_yz = hit_yz;
        cx.hit_idx = hit_idx;
        cx.bin_start = bin_start;
        cx.ro = row_offsets + (size_t)inst * g.R;
        cx.slab_base = inst * g.R;
        cx.z0 = grid_z0(g, inst);
        cx.s_rowx = s_rowx;
        const int32_t* ch = cand_hits + c * kCandMax;
        uint16_t* rowhit = tl_rowhit + c * g.RP;
        tl_nhits[c] = 0;  // overwritten at the end if a tracklet results
        // seed from hits 0, n/2, n-1
        const int i1 = n >> 1, i2 = n - 1;
        const float4 h0 = __ldg(&clusters[ch[0]]), h1 = __ldg(&clusters[ch[i1]]), h2 = __ldg(&clusters[ch[i2]]);
        // The state carries y and z relative to the first candidate hit.  The model is translation invariant in y
        // and z, so this is exact; it keeps the fp32 rounding of the two coordinates (ulp(20 cm), ulp(250 cm)) out
        // of q/pt and sinPhi, whose sensitivity to position noise is ~50/cm on 10-row tracklets.
        cx.yref = h0.y;
        cx.zref = h0.z;
        KfState st;
        if (!kf_seed(st, s_rowx[r0], 0.0f, 0.0f, s_rowx[r0 + i1], h1.y - cx.yref, s_rowx[r0 + i2], h2.y - cx.yref,
                     h2.z - cx.zref, g.cB, g.max_s, g.p0))
            continue;
        float chi2 = 0.0f;
        int nhits = 0;
        // phase A: the candidate's own hits ...
        bool ok = true;
        for (int i = 0; i < n; i++) {
            const int hg = ch[i];
            if (i > 0 && !kf_transport(st, s_rowx[r0 + i] - s_rowx[r0 + i - 1], g.cB, g.max_s)) {
                ok = false;
                break;
            }
            const float4 h = __ldg(&clusters[hg]);
            chi2 += kf_update(st, h.y - cx.yref, h.z - cx.zref, g.sy2, g.sz2);
            wc.transports += i > 0;
            wc.updates++;
            rowhit[r0 + i] = (uint16_t)(hg - cx.ro[r0 + i]);
            nhits++;
        }
        if (!ok) continue;
        // ... then upward pick-up
        int last_row = r0 + n - 1;
        const int r_top = follow_dir<+1>(g, cx, st, last_row, chi2, nhits, last_row, rowhit, nullptr, wc);
        // phase B: one step back to the start row (no update there), then downward pick-up
        if (!kf_transport(st, s_rowx[r0] - s_rowx[r_top], g.cB, g.max_s)) continue;
        wc.transports++;
        KfState rep = st;
        int first_row = r0;
        follow_dir<-1>(g, cx, st, r0, chi2, nhits, first_row, rowhit, &rep, wc);
        float* p = tl_par + c * 5;
        p[0] = rep.y + cx.yref; p[1] = rep.z + cx.zref; p[2] = rep.s; p[3] = rep.t; p[4] = rep.k;
        float* q = tl_cov + c * 15;
        q[0] = rep.c00; q[1] = rep.c10; q[2] = rep.c11; q[3] = rep.c20; q[4] = rep.c21; q[5] = rep.c22; q[6] = rep.c30;
        q[7] = rep.c31; q[8] = rep.c32; q[9] = rep.c33; q[10] = rep.c40; q[11] = rep.c41; q[12] = rep.c42;
        q[13] = rep.c43; q[14] = rep.c44;
        tl_chi2[c] = chi2;
        tl_rows[c] = first_row | (last_row << 8) | (first_row << 16);
        tl_nhits[c] = nhits;
    }
    // work counters: warp reduction, one atomic per warp and counter
    unsigned v[4] = {wc.transports, wc.updates, wc.examined, wc.searches};
#pragma unroll
    for (int q = 0; q < 4; q++) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], d);
        if ((threadIdx.x & 31) == 0 && v[q]) atomicAdd((unsigned long long*)&counts[6 + q], (unsigned long long)v[q]);
    }
}

int launch_follow(const DevGeom& g, const Workspace& w, const Problem& p, int n_sm, cudaStream_t s) {
    if (p.n_clusters == 0) return 0;
    // grid-stride over the (device-side) candidate count: enough CTAs to fill the machine, capped by the bound
    int64_t want = div_up(w.Cmax, kFollowThreads);
    int grid = (int)(want < (int64_t)n_sm * 16 ? want : (int64_t)n_sm * 16);
    if (grid < 1) grid = 1;
    follow_kernel<<<grid, kFollowThreads, 0, s>>>(g, p.clusters, p.row_offsets, w.hit_yz, w.hit_idx, w.bin_start,
                                                  w.cand_hits, w.cand_n, w.cand_slab, w.counts, w.Cmax, w.tl_par,
                                                  w.tl_cov, w.tl_chi2, w.tl_nhits, w.tl_rows, w.tl_rowhit);
    return 1;
}

}  // namespace tpc
