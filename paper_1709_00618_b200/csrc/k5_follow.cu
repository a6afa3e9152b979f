// S5: track following -- "fits track parameters to the track candidate and extrapolates the trajectory through the
// TPC sector volume to pick up additional clusters and refine the fit using a simplified Kalman filter"
// (Fig. 1c); constant Bz only.  Control flow: DESIGN.md "S5" (seed, phase A upward,
// one-step back transport, phase B downward).  One thread per candidate, all arithmetic fp32 in registers.
//
// Execution model: persistent warps, every lane a small state machine that advances its
// candidate by exactly ONE pad row per loop iteration whatever its phase (own hits / upward / back transport /
// downward), so the lanes of a warp run the same transport-search-update code instead of diverging on phase and
// track length.  A lane whose candidate has ended parks until a few lanes are parked, then those lanes write
// their tracklets and take new candidates from the warp's chunk of the device-wide queue (consecutive candidate
// ids start in neighbouring rows of one sector instance, which keeps the warp's loads in the same L1 lines).
#include "kf_math.cuh"

#ifndef TPC_FOLLOW_CTAS
#define TPC_FOLLOW_CTAS 6
#endif
namespace tpc {

constexpr int kFollowThreads = 128;
constexpr int kFollowCtasPerSm = TPC_FOLLOW_CTAS;
constexpr int kFollowChunk = 64;   // candidates a warp takes from the queue at a time
#ifndef TPC_FOLLOW_RELOAD
#define TPC_FOLLOW_RELOAD 4
#endif
constexpr int kFollowReload = TPC_FOLLOW_RELOAD;  // parked lanes that trigger a write-out / refill phase

enum FollowMode : int { kCand = 0, kUp = 1, kBack = 2, kDown = 3, kDone = 4, kIdle = 5 };

struct FollowArgs {
    const int32_t* row_offsets;
    const float2* hit_yz;
    const uint16_t* hit_idx;
    const uint16_t* bin_start;
    const int32_t* cand_hits;
    const int32_t* cand_n;
    const int32_t* cand_slab;
    int64_t* counts;
    int64_t Cmax;
    float* tl_par;
    float* tl_cov;
    float* tl_chi2;
    int32_t* tl_nhits;
    int32_t* tl_rows;
    uint16_t* tl_rowhit;
    uint32_t* tl_sel;  // S6 record of the tracklet (k6_select.cu), zeroed here
};

// The best hit of the pick-up search so far.
struct PickBest {
    int j;       // sorted position of the best hit, -1 = none
    float d2, y, z;
};

// Exact tie between two hits of the search (only duplicated clusters produce one): the lowest local index wins.
__device__ __noinline__ bool tie_lower_index(const uint16_t* __restrict__ idx, unsigned ja, unsigned jb) {
    return idx[ja] < idx[jb];
}

// One hit of the pick-up search: inside the gate and nearer than the best so far?  Ties -> lowest local index.
// The decision arithmetic is individually rounded fp32 (both sides decide in fp32).
__device__ __forceinline__ void pick_consider(PickBest& b, const uint16_t* __restrict__ idx, unsigned rb, int j,
                                              bool valid, float2 h, float yp, float zp, float wy, float wz) {
    const float dy = __fsub_rn(h.x, yp), dz = __fsub_rn(h.y, zp);
    const float d2 = __fadd_rn(__fmul_rn(dy, dy), __fmul_rn(dz, dz));
    const bool in = valid && fabsf(dy) <= wy && fabsf(dz) <= wz;
    bool better = in && d2 < b.d2;
    if (in && d2 == b.d2 && j != b.j) better = tie_lower_index(idx, rb + (unsigned)j, rb + (unsigned)b.j);
    if (better) {
        b.j = j;
        b.d2 = d2;
        b.y = h.x;
        b.z = h.y;
    }
}

__device__ __forceinline__ float sqrt_fast(float x) {  // x > 0, normal range
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

__device__ __forceinline__ void store_report(float4 (*s_rep)[kFollowThreads], const KfState& st) {
    s_rep[0][threadIdx.x] = make_float4(st.y, st.z, st.s, st.t);
    s_rep[1][threadIdx.x] = make_float4(st.k, st.c00, st.c10, st.c11);
    s_rep[2][threadIdx.x] = make_float4(st.c20, st.c21, st.c22, st.c30);
    s_rep[3][threadIdx.x] = make_float4(st.c31, st.c32, st.c33, st.c40);
    s_rep[4][threadIdx.x] = make_float4(st.c41, st.c42, st.c43, st.c44);
}

__device__ __forceinline__ void zero_report(float4 (*s_rep)[kFollowThreads]) {
#pragma unroll
    for (int q = 0; q < 5; q++) s_rep[q][threadIdx.x] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
}

// kCount: also accumulate the work counters counts[6..9] (roofline arithmetic; tpc_set_work_counters).  They are a
// property of the input, so the timed runs use the variant without them.
template <bool kCount>
__global__ void __launch_bounds__(kFollowThreads, kFollowCtasPerSm)
follow_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ FollowArgs a) {
    __shared__ float s_rowx[kMaxRows + 1];
    __shared__ float2 s_rowy[kMaxRows + 1];      // (y0, strips per cm) of the row's grid
    __shared__ float4 s_rep[5][kFollowThreads];  // reported state of the lane's tracklet (see kDown below)
    for (int q = threadIdx.x; q < g.R; q += kFollowThreads) {
        s_rowx[q] = g.row_x[q];
        s_rowy[q] = make_float2(g.row_y0[q], g.row_inv_sy[q]);
    }
    __syncthreads();
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const int n_cand = (int)min(a.counts[1], a.Cmax);
    unsigned long long* queue = reinterpret_cast<unsigned long long*>(&a.counts[10]);
    int wn = 0, we = 0;  // the warp's chunk [wn, we) of candidate ids (warp-uniform)
    bool exhausted = false;
    unsigned n_tr = 0, n_up = 0, n_ex = 0, n_se = 0;  // work counters (kCount only)

    // lane state
    int mode = kIdle;
    int c = 0, slab_base = 0;
    int r = 0, rn = 0, rb = 0;      // row of the state, row of the coming step and its offset in the hit arrays
    int r0 = 0, n = 0, i = 0;       // start row, candidate length, next own hit
    int hsn = 0;                    // sorted global position of the candidate's next own hit
    int nhits = 0, gap = 0, first_row = 0, last_row = 0;
    float yref = 0.0f, zref = 0.0f, z0 = 0.0f, chi2 = 0.0f;
    KfState st = {};

    for (;;) {
        unsigned act = __ballot_sync(full, mode < kDone);
        if (act == 0u || (!exhausted && 32 - __popc(act) >= kFollowReload)) {
            // ---- write-out of ended candidates ----
            if (mode == kDone) {
                const float4 q0 = s_rep[0][threadIdx.x], q1 = s_rep[1][threadIdx.x], q2 = s_rep[2][threadIdx.x],
                             q3 = s_rep[3][threadIdx.x], q4 = s_rep[4][threadIdx.x];
                float* p = a.tl_par + (size_t)c * 5;
                p[0] = q0.x + yref; p[1] = q0.y + zref; p[2] = q0.z; p[3] = q0.w; p[4] = q1.x;
                float* q = a.tl_cov + (size_t)c * 15;
                q[0] = q1.y; q[1] = q1.z; q[2] = q1.w; q[3] = q2.x; q[4] = q2.y; q[5] = q2.z; q[6] = q2.w;
                q[7] = q3.x; q[8] = q3.y; q[9] = q3.z; q[10] = q3.w; q[11] = q4.x; q[12] = q4.y; q[13] = q4.z;
                q[14] = q4.w;
                a.tl_chi2[c] = chi2;
                a.tl_rows[c] = first_row | (last_row << 8) | (first_row << 16);
                a.tl_nhits[c] = nhits;
                uint4* rec = reinterpret_cast<uint4*>(a.tl_sel + (size_t)c * g.sel_stride);
                for (int q4i = 0; q4i < g.sel_stride / 4; q4i++) rec[q4i] = make_uint4(0u, 0u, 0u, 0u);
                mode = kIdle;
            }
            // ---- refill ----
            if (!exhausted) {
                if (wn == we) {
                    unsigned long long v = 0;
                    if (lane == 0) v = atomicAdd(queue, (unsigned long long)kFollowChunk);
                    v = __shfl_sync(full, v, 0);
                    if (v >= (unsigned long long)n_cand) {
                        exhausted = true;
                    } else {
                        wn = (int)v;
                        we = min(wn + kFollowChunk, n_cand);
                    }
                }
                const unsigned idle = __ballot_sync(full, mode == kIdle);
                const int mine = wn + __popc(idle & ((1u << lane) - 1u));
                if (mode == kIdle && mine < we) {
                    c = mine;
                    const int slab0 = a.cand_slab[c];
                    const int inst = slab0 / g.R;
                    r0 = slab0 - inst * g.R;
                    n = a.cand_n[c];
                    slab_base = inst * g.R;
                    z0 = grid_z0(g, inst);
                    const int32_t* ch = a.cand_hits + (size_t)c * kCandMax;
                    // seed from hits 0, n/2, n-1
                    const int i1 = n >> 1, i2 = n - 1;
                    hsn = ch[0];
                    const float2 h0 = a.hit_yz[hsn], h1 = a.hit_yz[ch[i1]], h2 = a.hit_yz[ch[i2]];  // (y, z)
                    rb = a.row_offsets[slab_base + r0];
                    // The state carries y and z relative to the first candidate hit.  The model is translation
                    // invariant in y and z, so this is exact; it keeps the fp32 rounding of the two coordinates
                    // (ulp(20 cm), ulp(250 cm)) out of q/pt and sinPhi, whose sensitivity to position noise is
                    // ~50/cm on 10-row tracklets.
                    yref = h0.x;
                    zref = h0.y;
                    if (kf_seed(st, s_rowx[r0], 0.0f, 0.0f, s_rowx[r0 + i1], h1.x - yref, s_rowx[r0 + i2], h2.x - yref,
                                h2.y - zref, g.cB, g.max_s, g.p0)) {
                        mode = kCand;
                        i = 0;
                        r = rn = r0;
                        chi2 = 0.0f;
                        nhits = 0;
                        gap = 0;
                        first_row = r0;
                        last_row = r0;
                    } else {  // no tracklet: an all-zero record
                        nhits = 0;
                        chi2 = yref = zref = 0.0f;
                        first_row = last_row = 0;
                        zero_report(s_rep);
                        mode = kDone;
                    }
                }
                wn = min(we, wn + __popc(idle));
            }
            act = __ballot_sync(full, mode < kDone);
            if (act == 0u && exhausted) break;
        }
        if (mode < kDone) {
            // ---- one pad row: transport to row rn (offset rb), attach a hit, decide where to go next ----
            bool alive = true;
            float2 hc = make_float2(0.0f, 0.0f);
            if (mode == kCand) hc = a.hit_yz[hsn];  // issued before the transport arithmetic
            if (rn != r) {
                if (kf_transport(st, s_rowx[rn] - s_rowx[r], g.cB, g.max_s)) {
                    if (kCount) n_tr++;
                    r = rn;
                } else {
                    alive = false;
                    if (mode == kUp) {
                        mode = kBack;
                    } else if (mode == kDown) {
                        mode = kDone;
                    } else {  // inside the candidate's own hits, or the back transport: no tracklet
                        nhits = 0;
                        chi2 = yref = zref = 0.0f;
                        first_row = last_row = 0;
                        zero_report(s_rep);
                        mode = kDone;
                    }
                }
            }
            if (alive && mode == kBack) {
                // phase B starts: the reported state is the back-transported one until a hit is attached
                mode = r0 > 0 ? kDown : kDone;
                gap = 0;
                store_report(s_rep, st);
                alive = false;
            }
            if (alive) {
                float ym = hc.x, zm = hc.y;
                int li = hsn - rb;  // position of the hit to attach in the sorted row
                bool stop = false;
                if (mode != kCand) {
                    const float yp = st.y + yref, zp = st.z + zref;
                    if (fabsf(yp) > fmaf(s_rowx[r], g.tan_half, g.edge_margin)) {
                        stop = true;
                        alive = false;
                    } else {
                        // gate: 4 sigma of the predicted residual, capped (sigma > 0: tpc_tracker_create)
                        const float wy = fminf(g.wmax, g.gate * sqrt_fast(st.c00 + g.sy2));
                        const float wz = fminf(g.wmax, g.gate * sqrt_fast(st.c11 + g.sz2));
                        // The cells visited are a superset of the rounded fp32 gate test (margin m, monotone bins).
                        const float m = 1e-3f;
                        const float2 gy = s_rowy[r];
                        const int zb0 = zbin(zp - wz - m, z0, g.inv_cz, g.nz), zb1 = zbin(zp + wz + m, z0, g.inv_cz, g.nz);
                        const int ys0 = ybin(yp - wy - m, gy.x, gy.y, g.ny), ys1 = ybin(yp + wy + m, gy.x, gy.y, g.ny) + 1;
                        // one index per table entry (32-bit arithmetic, one wide multiply-add per address)
                        const unsigned tb0 = (unsigned)(slab_base + r) * (unsigned)g.nzp;
                        const unsigned ia = tb0 + (unsigned)(zb0 * g.ny), ib = tb0 + (unsigned)(zb1 * g.ny);
                        const int ja0 = a.bin_start[ia + ys0], ja1 = a.bin_start[ia + ys1];
                        int jb0 = 0, jb1 = 0;
                        if (zb1 > zb0) {
                            jb0 = a.bin_start[ib + ys0];
                            jb1 = a.bin_start[ib + ys1];
                        }
                        const int na = ja1 - ja0, nt = na + (jb1 - jb0);
                        if (kCount) {
                            n_se++;
                            n_ex += nt;
                        }
                        // The two ranges form one sequence k = 0..nt-1.  Its first two hits are examined in line
                        // (most searches see one or two); the loop below takes the rest one by one.
                        const int d = jb0 - na;  // position of sequence element k >= na is k + d
                        const int j0 = na > 0 ? ja0 : jb0;
                        const int j1 = na > 1 ? ja0 + 1 : 1 + d;
                        const unsigned urb = (unsigned)rb;
                        const float2 h0 = a.hit_yz[urb + (unsigned)(nt > 0 ? j0 : 0)];
                        const float2 h1 = a.hit_yz[urb + (unsigned)(nt > 1 ? j1 : 0)];
                        PickBest b{-1, __int_as_float(0x7f800000), 0.0f, 0.0f};
                        pick_consider(b, a.hit_idx, urb, j0, nt > 0, h0, yp, zp, wy, wz);
                        pick_consider(b, a.hit_idx, urb, j1, nt > 1, h1, yp, zp, wy, wz);
                        for (int k = 2; k < nt; k++) {
                            const int j = k < na ? ja0 + k : k + d;
                            pick_consider(b, a.hit_idx, urb, j, true, a.hit_yz[urb + (unsigned)j], yp, zp, wy, wz);
                        }
                        // z bins in between exist only when the cells are narrower than the gate (non-default grid_cell_z)
                        for (int zb = zb0 + 1; zb < zb1; zb++) {
                            const unsigned im = tb0 + (unsigned)(zb * g.ny);
                            const int jm0 = a.bin_start[im + ys0], jm1 = a.bin_start[im + ys1];
                            if (kCount) n_ex += jm1 - jm0;
                            for (int j = jm0; j < jm1; j++)
                                pick_consider(b, a.hit_idx, urb, j, true, a.hit_yz[urb + (unsigned)j], yp, zp, wy, wz);
                        }
                        ym = b.y;
                        zm = b.z;
                        li = b.j;
                    }
                }
                if (alive) {
                    const unsigned ih = (unsigned)c * (unsigned)g.RP + (unsigned)r;
                    __stcs(&a.tl_rowhit[ih], (uint16_t)li);  // li = -1 stores kNoHit
                    if (li >= 0) {
                        chi2 += kf_update(st, ym - yref, zm - zref, g.sy2, g.sz2);
                        if (kCount) n_up++;
                        nhits++;
                        gap = 0;
                        if (mode == kDown) {
                            first_row = r;
                            store_report(s_rep, st);
                        } else {
                            last_row = r;
                        }
                    } else if (++gap > g.max_gap) {
                        stop = true;
                    }
                }
                // where the next iteration goes
                if (mode == kCand) {
                    if (++i == n) mode = kUp;
                }
                if (mode == kUp) {
                    if (stop || r + 1 >= g.R) mode = kBack;
                } else if (mode == kDown) {
                    if (stop || r == 0) mode = kDone;
                }
            }
            // ---- set up the next step: its row, the row's offset, the candidate's next own hit ----
            if (mode < kDone) {
                rn = mode == kBack ? r0 : (mode == kDown ? r - 1 : (mode == kCand ? r0 + i : r + 1));
                rb = a.row_offsets[slab_base + rn];
                if (mode == kCand) hsn = a.cand_hits[(unsigned)c * (unsigned)kCandMax + (unsigned)i];
            }
        }
    }
    if (kCount) {  // work counters: warp reduction, one atomic per warp and counter
        unsigned v[4] = {n_tr, n_up, n_ex, n_se};
#pragma unroll
        for (int q = 0; q < 4; q++) {
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) v[q] += __shfl_xor_sync(full, v[q], d);
            if (lane == 0 && v[q]) atomicAdd((unsigned long long*)&a.counts[6 + q], (unsigned long long)v[q]);
        }
    }
}

int launch_follow(const DevGeom& g, const Workspace& w, const Problem& p, int n_sm, bool count_work, cudaStream_t s) {
    if (p.n_clusters == 0) return 0;
    // persistent grid: every SM holds kFollowCtasPerSm CTAs, capped by the candidate bound
    int64_t want = div_up(w.Cmax, kFollowThreads);
    int grid = (int)(want < (int64_t)n_sm * kFollowCtasPerSm ? want : (int64_t)n_sm * kFollowCtasPerSm);
    if (grid < 1) grid = 1;
    FollowArgs a{p.row_offsets, w.hit_yz, w.hit_idx, w.bin_start, w.cand_hits, w.cand_n, w.cand_slab,
                 w.counts,   w.Cmax,        w.tl_par, w.tl_cov,  w.tl_chi2,   w.tl_nhits,  w.tl_rows, w.tl_rowhit,
                 w.tl_sel};
    if (count_work)
        follow_kernel<true><<<grid, kFollowThreads, 0, s>>>(g, a);
    else
        follow_kernel<false><<<grid, kFollowThreads, 0, s>>>(g, a);
    return 1;
}

}  // namespace tpc
