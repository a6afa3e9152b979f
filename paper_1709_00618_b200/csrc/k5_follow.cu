// S5: track following -- "fits track parameters to the track candidate and extrapolates the trajectory through the
// TPC sector volume to pick up additional clusters and refine the fit using a simplified Kalman filter"
// (Fig. 1c); constant Bz only.  Control flow: DESIGN.md "S5" (seed, phase A upward,
// one-step back transport, phase B downward).  One thread per candidate, all arithmetic fp32 in registers.
//
// Two kernels:
//  * fit_candidates_kernel: the S4 chain walk (<= 9 dependent link loads), then seed + Kalman fit of the candidate's
//    own 4..10 hits, which wait in a per-thread column of shared memory; the state after the last own hit goes to
//    tl_state.
//  * follow_kernel: the row-by-row extrapolation.  Persistent warps, every lane a small state machine that advances
//    its candidate by ONE pad row per loop iteration (upward / back transport / downward), with the lanes refilled
//    from a device-wide queue as candidates end.  A pick-up search reads the cell-table entries of the exact gate
//    window and then the window's first hits, all loads of a kind in flight together; examining a superset of cells
//    is harmless because every hit still passes the exact gate test (the grid is an acceleration structure only).
//    The 20 filter values and what every step touches live in registers (64: eight CTAs per SM), what a step touches
//    at most once in shared memory.  (Variants measured and rejected -- speculative loads, prefetches, buffered
//    stores, an asynchronous candidate supply -- are listed in DESIGN.md section 5.)
#include "kf_math.cuh"

#ifndef TPC_FOLLOW_CTAS
#define TPC_FOLLOW_CTAS 8
#endif
#ifndef TPC_FOLLOW_RELOAD
#define TPC_FOLLOW_RELOAD 6
#endif
namespace tpc {

constexpr int kFollowThreads = 128;
constexpr int kFollowCtasPerSm = TPC_FOLLOW_CTAS;
#ifndef TPC_FOLLOW_CHUNK
#define TPC_FOLLOW_CHUNK 0
#endif
constexpr int kFollowChunk = TPC_FOLLOW_CHUNK;  // candidates a warp takes from the queue at a time; 0 = as many as it has idle lanes
constexpr int kFollowReload = TPC_FOLLOW_RELOAD;  // parked lanes that trigger a write-out / refill phase
constexpr int kFitThreads = 128;
#ifndef TPC_DIRECT_HITS
#define TPC_DIRECT_HITS 4
#endif

constexpr int kDirectHits = TPC_DIRECT_HITS;      // hits of a window examined in line (the rest in a loop)
constexpr float kCellMargin = 1e-3f;  // [cm] the visited cells are a superset of the rounded fp32 gate test

enum FollowMode : int { kUp = 0, kBack = 1, kDown = 2, kDone = 3, kIdle = 4 };

struct FollowArgs {
    const int32_t* row_offsets;
    const float2* hit_yz;
    const uint16_t* hit_idx;
    const uint16_t* bin_start;
    const int32_t* up;          // cleaned up-links (sorted space)
    const int32_t* cand_start;  // sorted global position of the candidate's start hit
    const int32_t* cand_slab;
    int32_t* usr_cand_hits;     // optional user-facing S4 outputs (input-order global indices), NULL = skip
    int32_t* usr_cand_n;
    int64_t usr_cand_cap;
    int64_t* counts;
    int64_t Cmax;
    float4* tl_state;  // [6][Cmax] state after the candidate's own hits (fit kernel -> follow kernel)
    float* tl_par;
    float* tl_cov;
    float* tl_chi2;
    int32_t* tl_nhits;
    int32_t* tl_rows;
    uint16_t* tl_rowhit;
    uint32_t* tl_sel;  // S6 record of the tracklet (k6_select.cu), zeroed here
};

__device__ __forceinline__ void zero_tracklet(const DevGeom& g, const FollowArgs& a, int c) {
    float* p = a.tl_par + (size_t)c * 5;
#pragma unroll
    for (int q = 0; q < 5; q++) p[q] = 0.0f;
    float* v = a.tl_cov + (size_t)c * 15;
#pragma unroll
    for (int q = 0; q < 15; q++) v[q] = 0.0f;
    a.tl_chi2[c] = 0.0f;
    a.tl_rows[c] = 0;
    a.tl_nhits[c] = 0;
    uint4* rec = reinterpret_cast<uint4*>(a.tl_sel + (size_t)c * g.sel_stride);
    for (int q = 0; q < g.sel_stride / 4; q++) rec[q] = make_uint4(0u, 0u, 0u, 0u);
}

// ---- fit of the candidate's own hits -----------------------------------------------------------------------------
// The candidate's hits are staged per thread in shared memory ([hit][thread]: conflict-free) instead of register
// arrays: the kernel is bound by the latency of the chain walk (9 dependent loads per thread), and at ~60 registers
// twice as many warps are resident to hide it as with the hits in registers (104).
#ifndef TPC_FIT_CTAS
#define TPC_FIT_CTAS 8
#endif
template <bool kCount>
__global__ void __launch_bounds__(kFitThreads, TPC_FIT_CTAS)
fit_candidates_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ FollowArgs a) {
    __shared__ float2 s_h[kCandMax][kFitThreads];      // (y, z) of the candidate's q-th hit
    __shared__ unsigned s_loc[kCandMax][kFitThreads];  // its position in the sorted row | pad row << 16
    const int n_cand = (int)min(a.counts[1], a.Cmax);
    const int t = threadIdx.x;
    unsigned n_tr = 0, n_up = 0;
    // grid-stride: the candidate count is only known on the device, and a grid sized by its bound (N / 4) would be
    // four fifths empty CTAs
    for (int c = blockIdx.x * kFitThreads + t; c < n_cand; c += gridDim.x * kFitThreads) {
        const int slab0 = a.cand_slab[c];
        const int inst = slab0 / g.R;
        const int r0 = slab0 - inst * g.R;
        const int slab_base0 = slab0 - r0;
        const bool usr = a.usr_cand_hits && c < a.usr_cand_cap;  // parity/user copy: input-order global indices
        // S4 concatenation: the candidate's hits are the first <= cand_max hits of the chain of up-links that
        // starts at its start hit (sorted global positions); the walk is 9 dependent 4-byte loads per thread.
        // Consecutive pad rows, or one row skipped where S2 bridged a missing row (A2').
        int n = 0, row = r0, rbq = a.row_offsets[slab0];
        int pos = a.cand_start[c];
#pragma unroll 1
        for (int q = 0; q < kCandMax && q < g.cand_max && pos >= 0; q++) {
            if (q > 0) {
                row++;
                rbq = a.row_offsets[slab_base0 + row];
                if (g.bridge) {
                    const int nb2 = a.row_offsets[slab_base0 + row + 1];  // row + 1 <= R: a valid entry
                    if (pos >= nb2) {
                        row++;
                        rbq = nb2;
                    }
                }
            }
            const int nxt = a.up[pos];  // next link first: the only dependent load of the walk
            s_h[q][t] = a.hit_yz[pos];
            s_loc[q][t] = (unsigned)(pos - rbq) | ((unsigned)row << 16);
            if (usr) a.usr_cand_hits[(size_t)c * kCandMax + q] = rbq + (int)a.hit_idx[pos];
            pos = nxt;
            n = q + 1;
        }
        if (usr)
            for (int q = n; q < kCandMax; q++) a.usr_cand_hits[(size_t)c * kCandMax + q] = -1;
        if (a.usr_cand_n && c < a.usr_cand_cap) a.usr_cand_n[c] = n;
        // seed from hits 0, n/2, n-1.  The state carries y and z relative to the last attached hit: the model is
        // translation invariant in y and z, so this is exact, and it keeps the fp32 rounding of the two
        // coordinates (ulp(20 cm), ulp(250 cm)) out of the state.
        const int i1 = n >> 1, i2 = n - 1;
        const float2 h0 = s_h[0][t], h1 = s_h[i1][t], h2 = s_h[i2][t];
        const float x0 = g.row_x[r0], x1 = g.row_x[s_loc[i1][t] >> 16], x2 = g.row_x[s_loc[i2][t] >> 16];
        float yref = h0.x, zref = h0.y;
        KfState st;
        bool ok = kf_seed(st, x0, 0.0f, 0.0f, x1, h1.x - yref, x2, h2.x - yref, h2.y - zref, g.cB, g.max_s, g.p0);
        float chi2 = 0.0f;
        if (ok) {
            float xp = x0;
#pragma unroll 1
            for (int q = 0; q < n && ok; q++) {
                const float2 h = s_h[q][t];
                if (q > 0) {
                    const float x = g.row_x[s_loc[q][t] >> 16];
                    ok = kf_transport(st, x - xp, g.cB, g.max_s);
                    xp = x;
                    if (kCount && ok) n_tr++;
                }
                if (ok) {
                    chi2 += kf_update(st, h.x - yref, h.y - zref, g.sy2, g.sz2);
                    yref = h.x;  // the state's (y, z) frame follows the attached hit (kf_update)
                    zref = h.y;
                    if (kCount) n_up++;
                }
            }
        }
        float4* ts = a.tl_state + c;
        const size_t cs = (size_t)a.Cmax;
        if (ok) {
            ts[0] = make_float4(st.y, st.z, st.s, st.t);
            ts[cs] = make_float4(st.k, st.c00, st.c10, st.c11);
            ts[2 * cs] = make_float4(st.c20, st.c21, st.c22, st.c30);
            ts[3 * cs] = make_float4(st.c31, st.c32, st.c33, st.c40);
            ts[4 * cs] = make_float4(st.c41, st.c42, st.c43, st.c44);
            uint16_t* rh = a.tl_rowhit + (size_t)c * g.RP;
            int prev = r0;
            for (int q = 0; q < n; q++) {
                const unsigned loc = s_loc[q][t];
                const int rq = (int)(loc >> 16);
                __stcs(&rh[rq], (uint16_t)(loc & 0xffffu));
                if (rq - prev == 2) __stcs(&rh[rq - 1], kNoHit);  // the bridged row
                prev = rq;
            }
            // own hits | (last own row - start row) << 8
            ts[5 * cs] = make_float4(yref, zref, chi2, __int_as_float(n | ((prev - r0) << 8)));
        } else {  // no tracklet: an all-zero record, and the follower skips the candidate
            ts[5 * cs] = make_float4(0.0f, 0.0f, 0.0f, __int_as_float(0));
            zero_tracklet(g, a, c);
        }
    }
    if (kCount) {
        const unsigned full = 0xffffffffu;
        n_tr = __reduce_add_sync(full, n_tr);
        n_up = __reduce_add_sync(full, n_up);
        if ((threadIdx.x & 31) == 0) {
            if (n_tr) atomicAdd((unsigned long long*)&a.counts[6], (unsigned long long)n_tr);
            if (n_up) atomicAdd((unsigned long long*)&a.counts[7], (unsigned long long)n_up);
            if (n_tr) atomicAdd((unsigned long long*)&a.counts[11], (unsigned long long)n_tr);
            if (n_up) atomicAdd((unsigned long long*)&a.counts[12], (unsigned long long)n_up);
        }
    }
}

// ---- row-by-row following ------------------------------------------------------------------------------------------

// The best hit of the pick-up search so far, and whether an exact tie for the best distance was seen on the way.
struct PickBest {
    int j;       // sorted position (in its row) of the best hit, -1 = none
    float d2, y, z;
    bool tie;
};

// One hit of the pick-up search: inside the gate and nearer than the best so far?  The decision arithmetic is
// individually rounded fp32 (both sides decide in fp32).  Strictly-nearer wins here; an exact tie for
// the best distance (only duplicated clusters produce one) is only RECORDED, and the search is then redone out of
// line by pick_exact with the full rule (lowest local index).  A tie for the minimum is always seen: the second of
// two equal-best hits meets either the first or something nearer still.
__device__ __forceinline__ void pick_consider(PickBest& b, int j, bool valid, float2 h, float yp, float zp, float wy,
                                              float wz) {
    const float dy = __fsub_rn(h.x, yp), dz = __fsub_rn(h.y, zp);
    const float d2 = __fadd_rn(__fmul_rn(dy, dy), __fmul_rn(dz, dz));
    const bool in = valid && fabsf(dy) <= wy && fabsf(dz) <= wz;
    const bool better = in && d2 < b.d2;
    b.tie = b.tie || (in && d2 == b.d2);
    b.j = better ? j : b.j;
    b.d2 = better ? d2 : b.d2;
    b.y = better ? h.x : b.y;
    b.z = better ? h.y : b.z;
}

// The whole pick-up search of one row with the complete rule: nearest hit inside the gate by (dy^2 + dz^2), ties ->
// lowest local index.  tb = the row's cell table, rowh / rowi = the row's sorted hits and their local indices.
__device__ __noinline__ int pick_exact(const uint16_t* __restrict__ tb, const float2* __restrict__ rowh,
                                       const uint16_t* __restrict__ rowi, int ny, int zb0, int zb1, int ys0, int ys1,
                                       float yp, float zp, float wy, float wz) {
    int bj = -1;
    float bd2 = __int_as_float(0x7f800000);
    unsigned bi = 0u;
    for (int zb = zb0; zb <= zb1; zb++) {
        const uint16_t* t = tb + zb * ny;
        const int j1 = t[ys1];
        for (int j = t[ys0]; j < j1; j++) {
            const float2 h = rowh[j];
            const float dy = __fsub_rn(h.x, yp), dz = __fsub_rn(h.y, zp);
            if (!(fabsf(dy) <= wy && fabsf(dz) <= wz)) continue;
            const float d2 = __fadd_rn(__fmul_rn(dy, dy), __fmul_rn(dz, dz));
            const unsigned li = rowi[j];
            if (d2 < bd2 || (d2 == bd2 && li < bi)) {
                bd2 = d2;
                bi = li;
                bj = j;
            }
        }
    }
    return bj;
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

// The window's hits as one sequence of nt sorted positions: element k < na sits at k + ja0, element k >= na at k + d.
struct HitSeq {
    int ja0, na, nt, d;
};

__device__ __forceinline__ HitSeq hit_seq(unsigned t00, unsigned t01, unsigned t10, unsigned t11, bool two) {
    HitSeq s;
    s.ja0 = (int)t00;
    s.na = (int)t01 - (int)t00;
    s.nt = s.na + (two ? (int)t11 - (int)t10 : 0);
    s.d = (int)t10 - s.na;
    return s;
}

// kCount: also accumulate the work counters counts[6..9] (roofline arithmetic; tpc_set_work_counters).  They are a
// property of the input, so the timed runs use the variant without them.
template <bool kCount>
__global__ void __launch_bounds__(kFollowThreads, kFollowCtasPerSm)
follow_kernel(const __grid_constant__ DevGeom g, const __grid_constant__ FollowArgs a) {
    // per row: x, lower edge of the y grid, strips per cm, |y| limit of the sector (x tan(half angle) + margin)
    __shared__ float4 s_row[kMaxRows + 1];
    __shared__ float4 s_rep[5][kFollowThreads];  // reported state of the lane's tracklet (see kDown below)
    // values touched only in the write-out / refill phase live in shared memory, not in registers of the row loop
    __shared__ int s_cand[kFollowThreads];        // the lane's candidate id
    __shared__ int2 s_chunk[kFollowThreads / 32];  // the warp's chunk [x, y) of candidate ids
    // lane state that is read or written once per row at most: kept out of the register file so that
    // kFollowCtasPerSm CTAs fit (the step is bound by load latency: resident warps count)
    __shared__ float s_z0[kFollowThreads], s_chi2[kFollowThreads];
    __shared__ int s_r0[kFollowThreads], s_first[kFollowThreads], s_last[kFollowThreads];
    __shared__ uint16_t* s_rh[kFollowThreads];  // the candidate's row-indexed hit table
    if (threadIdx.x < kFollowThreads / 32) s_chunk[threadIdx.x] = make_int2(0, 0);
    for (int q = threadIdx.x; q < g.R; q += kFollowThreads) {
        const float x = g.row_x[q];
        s_row[q] = make_float4(x, g.row_y0[q], g.row_inv_sy[q], fmaf(x, g.tan_half, g.edge_margin));
    }
    __syncthreads();
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const unsigned tab_stride = (unsigned)g.nzp >> 4;  // cell-table row in units of 16 entries (nzp is a multiple)
    bool exhausted = false;
    unsigned n_tr = 0, n_up = 0, n_ex = 0, n_se = 0;  // work counters (kCount only)

    // lane state
    int mode = kIdle;
    int slab_base = 0;
    int r = 0, rn = 0;  // row of the state, row of the coming step
    int nhits = 0, gap = 0;
    float yref = 0.0f, zref = 0.0f;
    float xr = 0.0f;  // x of row r
    KfState st = {};
    int rb_next = 0;  // offset of row rn (loaded one step ahead)

    for (;;) {
        unsigned act = __ballot_sync(full, mode < kDone);
        if (act == 0u || (!exhausted && 32 - __popc(act) >= kFollowReload)) {
            // ---- write-out of ended candidates ----
            if (mode == kDone) {
                const int c = s_cand[threadIdx.x];
                const float4 q0 = s_rep[0][threadIdx.x], q1 = s_rep[1][threadIdx.x], q2 = s_rep[2][threadIdx.x],
                             q3 = s_rep[3][threadIdx.x], q4 = s_rep[4][threadIdx.x];
                float* p = a.tl_par + (size_t)c * 5;
                p[0] = q0.x + yref; p[1] = q0.y + zref; p[2] = q0.z; p[3] = q0.w; p[4] = q1.x;
                float* q = a.tl_cov + (size_t)c * 15;
                q[0] = q1.y; q[1] = q1.z; q[2] = q1.w; q[3] = q2.x; q[4] = q2.y; q[5] = q2.z; q[6] = q2.w;
                q[7] = q3.x; q[8] = q3.y; q[9] = q3.z; q[10] = q3.w; q[11] = q4.x; q[12] = q4.y; q[13] = q4.z;
                q[14] = q4.w;
                a.tl_chi2[c] = s_chi2[threadIdx.x];
                const int first_row = s_first[threadIdx.x];
                a.tl_rows[c] = first_row | (s_last[threadIdx.x] << 8) | (first_row << 16);
                a.tl_nhits[c] = nhits;
                uint4* rec = reinterpret_cast<uint4*>(a.tl_sel + (size_t)c * g.sel_stride);
                for (int q4i = 0; q4i < g.sel_stride / 4; q4i++) rec[q4i] = make_uint4(0u, 0u, 0u, 0u);
                mode = kIdle;
            }
            // ---- refill ----
            if (!exhausted) {
                const unsigned idle = __ballot_sync(full, mode == kIdle);
                const int n_cand = (int)min(a.counts[1], a.Cmax);
                const size_t cs = (size_t)a.Cmax;
                int wn = s_chunk[threadIdx.x >> 5].x, we = s_chunk[threadIdx.x >> 5].y;
                if (wn == we) {
                    // kFollowChunk = 0: take exactly as many ids as there are idle lanes (best balance at the end of
                    // the queue: no warp sits on ids it cannot start yet)
                    const int take = kFollowChunk > 0 ? kFollowChunk : __popc(idle);
                    unsigned long long v = 0;
                    if (lane == 0)
                        v = atomicAdd(reinterpret_cast<unsigned long long*>(&a.counts[10]), (unsigned long long)take);
                    v = __shfl_sync(full, v, 0);
                    if (v >= (unsigned long long)n_cand) {
                        exhausted = true;
                    } else {
                        wn = (int)v;
                        we = min(wn + take, n_cand);
                    }
                }
                const int mine = wn + __popc(idle & ((1u << lane) - 1u));
                if (mode == kIdle && mine < we) {
                    const int c = mine;
                    s_cand[threadIdx.x] = c;
                    const float4* ts = a.tl_state + c;
                    // all loads of the hand-over in flight together (one memory round trip, then row_offsets)
                    const float4 t5 = ts[5 * cs];
                    const float4 t0 = ts[0], t1 = ts[cs], t2 = ts[2 * cs], t3 = ts[3 * cs], t4 = ts[4 * cs];
                    const int slab0 = a.cand_slab[c];
                    const int nbits = __float_as_int(t5.w);  // own hits | (last own row - start row) << 8
                    const int n = nbits & 0xff;
                    if (n > 0) {  // n == 0: the fit of the candidate's own hits failed, nothing to follow
                        const int inst = slab0 / g.R;
                        const int r0 = slab0 - inst * g.R;
                        slab_base = inst * g.R;
                        s_r0[threadIdx.x] = r0;
                        s_z0[threadIdx.x] = grid_z0(g, inst);
                        st.y = t0.x; st.z = t0.y; st.s = t0.z; st.t = t0.w;
                        st.k = t1.x; st.c00 = t1.y; st.c10 = t1.z; st.c11 = t1.w;
                        st.c20 = t2.x; st.c21 = t2.y; st.c22 = t2.z; st.c30 = t2.w;
                        st.c31 = t3.x; st.c32 = t3.y; st.c33 = t3.z; st.c40 = t3.w;
                        st.c41 = t4.x; st.c42 = t4.y; st.c43 = t4.z; st.c44 = t4.w;
                        yref = t5.x;
                        zref = t5.y;
                        s_chi2[threadIdx.x] = t5.z;
                        nhits = n;
                        gap = 0;
                        s_first[threadIdx.x] = r0;
                        r = r0 + (nbits >> 8);
                        s_last[threadIdx.x] = r;
                        xr = s_row[r].x;
                        mode = r + 1 < g.R ? kUp : kBack;
                        rn = mode == kUp ? r + 1 : r0;
                        rb_next = a.row_offsets[slab_base + rn];
                        s_rh[threadIdx.x] = a.tl_rowhit + (size_t)c * (size_t)g.RP;
                    }
                }
                __syncwarp();
                if (lane == 0) s_chunk[threadIdx.x >> 5] = make_int2(min(we, wn + __popc(idle)), we);
                __syncwarp();
            }
            act = __ballot_sync(full, mode < kDone);
            if (act == 0u && exhausted) break;
        }
        if (mode < kDone) {
            // ---- one pad row: transport to row rn, attach a hit, decide where to go next.  Written as one
            // straight path with flags: the lanes of a warp differ in phase, and every branch taken by a few
            // lanes costs the whole warp its instructions.
            const bool is_back = mode == kBack;
            const bool down = mode == kDown;
            const float4 rd = s_row[rn];
            const bool t_ok = kf_transport(st, rd.x - xr, g.cB, g.max_s);
            if (kCount && t_ok) n_tr++;
            r = t_ok ? rn : r;
            xr = t_ok ? rd.x : xr;
            const float yp = st.y + yref, zp = st.z + zref;
            const bool inside = fabsf(yp) <= rd.w;
            const bool search = t_ok && !is_back && inside;
            bool hit = false;
            if (search) {
                // gate: 4 sigma of the predicted residual, capped (sigma > 0: tpc_tracker_create)
                const float wy = fminf(g.wmax, g.gate * sqrt_fast(st.c00 + g.sy2));
                const float wz = fminf(g.wmax, g.gate * sqrt_fast(st.c11 + g.sz2));
                // the cells of the gate window, widened by a margin so that they cover the rounded fp32 gate test
                const float my = wy + kCellMargin, mz = wz + kCellMargin;
                const float z0 = s_z0[threadIdx.x];
                const int zb0 = zbin(zp - mz, z0, g.inv_cz, g.nz), zb1 = zbin(zp + mz, z0, g.inv_cz, g.nz);
                const int ys0 = ybin(yp - my, rd.y, rd.z, g.ny), ys1 = ybin(yp + my, rd.y, rd.z, g.ny) + 1;
                // cell-table entries of the window (row index in 32-byte units: n_inst * R * nzp may exceed 2^32)
                const uint16_t* tb = a.bin_start + (size_t)((unsigned)(slab_base + r) * tab_stride) * 16u;
                const unsigned o0 = (unsigned)(zb0 * g.ny), o1 = (unsigned)(zb1 * g.ny);
                const bool two = zb1 > zb0;
                const unsigned t00 = tb[o0 + (unsigned)ys0], t01 = tb[o0 + (unsigned)ys1];
                unsigned t10 = 0u, t11 = 0u;
                if (two) {
                    t10 = tb[o1 + (unsigned)ys0];
                    t11 = tb[o1 + (unsigned)ys1];
                }
                const HitSeq q = hit_seq(t00, t01, t10, t11, two);
                if (kCount) {
                    n_se++;
                    n_ex += q.nt;
                }
                const unsigned urb = (unsigned)rb_next;  // hits of the row: a.hit_yz[urb + position], 32-bit index
                const float2* rowh = a.hit_yz + urb;
                // The window's hits form one sequence k = 0..nt-1.  The first kDirectHits are loaded together (one
                // memory round trip) and compared without a branch, the rest (few lanes) one by one.
                PickBest b{-1, __int_as_float(0x7f800000), 0.0f, 0.0f, false};
                {
                    float2 h[kDirectHits];
                    int j[kDirectHits];
#pragma unroll
                    for (int k = 0; k < kDirectHits; k++) {
                        j[k] = k + (k < q.na ? q.ja0 : q.d);
                        h[k] = make_float2(0.0f, 0.0f);
                        if (k < q.nt) h[k] = a.hit_yz[urb + (unsigned)j[k]];
                    }
#pragma unroll
                    for (int k = 0; k < kDirectHits; k++) pick_consider(b, j[k], k < q.nt, h[k], yp, zp, wy, wz);
                }
                for (int k = kDirectHits; k < q.nt; k++) {  // test the gate first, most of these hits fail it
                    const int j = k + (k < q.na ? q.ja0 : q.d);
                    const float2 h = a.hit_yz[urb + (unsigned)j];
                    if (fabsf(__fsub_rn(h.x, yp)) <= wy && fabsf(__fsub_rn(h.y, zp)) <= wz)
                        pick_consider(b, j, true, h, yp, zp, wy, wz);
                }
                // z bins in between exist only when the cells are narrower than the gate (non-default grid_cell_z)
                for (int zb = zb0 + 1; zb < zb1; zb++) {
                    const unsigned om = (unsigned)(zb * g.ny);
                    const int jm0 = tb[om + (unsigned)ys0], jm1 = tb[om + (unsigned)ys1];
                    if (kCount) n_ex += jm1 - jm0;
                    for (int j = jm0; j < jm1; j++) pick_consider(b, j, true, a.hit_yz[urb + (unsigned)j], yp, zp, wy, wz);
                }
                if (b.tie) {  // duplicated clusters: redo the search with the complete tie rule
                    b.j = pick_exact(tb, rowh, a.hit_idx + urb, g.ny, zb0, zb1, ys0, ys1, yp, zp, wy, wz);
                    const float2 h = a.hit_yz[urb + (unsigned)b.j];  // a tie was between hits inside the gate: b.j >= 0
                    b.y = h.x;
                    b.z = h.y;
                }
                // (Collecting 8 rows of the table in shared memory and storing them with one 16-byte request was
                // measured: 12.1 ms against 11.3 ms -- the 2-byte stores are not what limits the step.)
                __stcs(&s_rh[threadIdx.x][r], (uint16_t)b.j);  // -1 = kNoHit
                hit = b.j >= 0;
                if (hit) {
                    s_chi2[threadIdx.x] += kf_update(st, b.y - yref, b.z - zref, g.sy2, g.sz2);
                    (down ? s_first : s_last)[threadIdx.x] = r;
                    yref = b.y;  // the state's (y, z) frame follows the attached hit (kf_update)
                    zref = b.z;
                    if (kCount) n_up++;
                }
            }
            // bookkeeping of the step, as selects
            nhits += hit ? 1 : 0;
            gap = (hit || is_back) ? 0 : gap + (search ? 1 : 0);
            if ((hit && down) || (is_back && t_ok)) store_report(s_rep, st);  // reported state: see kDown / kBack
            // where to go next: up until the track stops or the detector ends, one step back to the start row, down
            const bool go_on = t_ok && inside && gap <= g.max_gap && (down ? r > 0 : r + 1 < g.R);
            const int after = down ? kDone : kBack;
            int next = go_on ? mode : after;
            if (is_back) {
                next = (t_ok && s_r0[threadIdx.x] > 0) ? kDown : kDone;
                if (!t_ok) {  // the back transport failed: no tracklet, an all-zero record
                    nhits = 0;
                    yref = zref = 0.0f;
                    s_chi2[threadIdx.x] = 0.0f;
                    s_first[threadIdx.x] = s_last[threadIdx.x] = 0;
#pragma unroll
                    for (int q = 0; q < 5; q++) s_rep[q][threadIdx.x] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                }
            }
            mode = next;
            rn = mode == kDown ? r - 1 : r + 1;
            if (mode == kBack) rn = s_r0[threadIdx.x];
            // offset of the coming row, one step ahead.  (Prefetching the next row's cell-table entries as well --
            // the same cell of row rn -- was measured twice and lost, +0.5 ms: the L1 data pipe is already half busy.)
            if (mode < kDone) rb_next = a.row_offsets[slab_base + rn];
        }
    }
    if (kCount) {  // work counters: warp reduction, one atomic per warp and counter
        unsigned v[4] = {n_tr, n_up, n_ex, n_se};
#pragma unroll
        for (int q = 0; q < 4; q++) {
            v[q] = __reduce_add_sync(full, v[q]);
            if (lane == 0 && v[q]) atomicAdd((unsigned long long*)&a.counts[6 + q], (unsigned long long)v[q]);
        }
    }
}

static FollowArgs follow_args(const Workspace& w, const Problem& p, const ChainOut& u) {
    return FollowArgs{p.row_offsets, w.hit_yz,  w.hit_idx,  w.bin_start, w.up,        w.cand_start, w.cand_slab,
                      u.cand_hits,   u.cand_n,  u.cand_cap, w.counts,    w.Cmax,      w.tl_state,   w.tl_par,
                      w.tl_cov,      w.tl_chi2, w.tl_nhits, w.tl_rows,   w.tl_rowhit, w.tl_sel};
}

int launch_fit(const DevGeom& g, const Workspace& w, const Problem& p, const ChainOut& u, bool count_work, cudaStream_t s) {
    if (p.n_clusters == 0) return 0;
    const FollowArgs a = follow_args(w, p, u);
    // the candidate count lives on the device: the grid is sized by its bound and bounded by it inside
    const int64_t want = div_up(w.Cmax, kFitThreads);
    const int grid = (int)(want < 148 * TPC_FIT_CTAS * 8 ? want : 148 * TPC_FIT_CTAS * 8);
    if (count_work)
        fit_candidates_kernel<true><<<grid, kFitThreads, 0, s>>>(g, a);
    else
        fit_candidates_kernel<false><<<grid, kFitThreads, 0, s>>>(g, a);
    return 1;
}

int launch_follow(const DevGeom& g, const Workspace& w, const Problem& p, int n_sm, bool count_work, cudaStream_t s) {
    if (p.n_clusters == 0) return 0;
    const FollowArgs a = follow_args(w, p, ChainOut{nullptr, 0, nullptr, nullptr, 0});
    // persistent grid: every SM holds kFollowCtasPerSm CTAs, capped by the candidate bound
    const int64_t want = div_up(w.Cmax, kFollowThreads);
    int grid = (int)(want < (int64_t)n_sm * kFollowCtasPerSm ? want : (int64_t)n_sm * kFollowCtasPerSm);
    if (grid < 1) grid = 1;
    if (count_work)
        follow_kernel<true><<<grid, kFollowThreads, 0, s>>>(g, a);
    else
        follow_kernel<false><<<grid, kFollowThreads, 0, s>>>(g, a);
    return 1;
}

}  // namespace tpc
