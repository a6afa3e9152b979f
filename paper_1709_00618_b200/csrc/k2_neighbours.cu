// S2: Cellular-Automaton neighbour finder -- "forming links of adjacent hits arranged close to a straight line"
// (Fig. 1a).  For every hit of row r the pair (u in row r+1, d in row r-1) inside the search window
// that minimises the squared second difference D, D <= d2max, ties broken by the lowest local cluster index
// (BASELINE.json north_star; DESIGN.md "S2" gives the exact evaluation order).
//
// Bit-exact contract with the oracle: every fp32 operation below is an explicitly rounded intrinsic
// (__fadd_rn/__fsub_rn/__fmul_rn are never contracted into FMAs), the window is a set of pure comparisons against
// pre-rounded bounds, and the minimum is taken over (D, u, d) lexicographically, so the result does not depend on
// the order in which the grid presents the hits.  This file is additionally compiled with -fmad=false.
//
// One CTA per (sector instance, pad row).  The sorted (y,z) and the cell tables of the rows it touches are brought
// into shared memory by 1-D bulk copies (TMA) completing on an mbarrier -- one elected thread issues them, nobody
// spends instructions on staging; rows or tables too long for the buffers are read in place.  Per hit the search is two flat loops: the window hits of row r-1 (a handful, through the 2-D grid) are
// collected in registers, then every window hit of row r+1 is paired with them.
#include "tpc_common.cuh"

namespace tpc {

#ifndef TPC_NB_THREADS
#define TPC_NB_THREADS 96  // measured: 64 -> 4.65, 96 -> 4.17, 128 -> 4.31, 192 -> 5.23, 256 -> 5.79 ms on the bench workload
#endif
constexpr int kNbThreads = TPC_NB_THREADS;
#ifndef TPC_NB_STAGE_HITS
#define TPC_NB_STAGE_HITS 382
#endif
constexpr int kNbStageHits = TPC_NB_STAGE_HITS;  // hits of one row that fit its shared-memory buffer (8 B each)
constexpr int kNbStageTbl = 4096;   // max table entries per row staged in shared memory (2 B each, two rows)
constexpr int kNbList = 4;          // window hits per neighbour row kept in registers; more -> exact slow path

struct RowView {
    const float2* yz;
    const uint16_t* idx;
    const uint16_t* tbl;
    float y0, inv_sy;
};

struct Best {
    float D;
    int ju, jd;  // positions in the sorted rows r+1 / r-1, -1 = none
};

// Exact tie of D between two admissible pairs (duplicated clusters only): the lower (local index of u, local index
// of d) wins.  Local indices = positions in the INPUT row segments, so the result does not depend on the sorted order.
__device__ __noinline__ bool tie_lower(const uint16_t* __restrict__ idx_up, const uint16_t* __restrict__ idx_dn, int ju,
                                       int jd, int bu, int bd) {
    const int iu = idx_up[ju], ibu = idx_up[bu];
    return iu < ibu || (iu == ibu && idx_dn[jd] < idx_dn[bd]);
}

// Keep the minimum over (D, local index of u, local index of d).  Straight-line code: `adm` says whether the pair
// exists and is admissible; b.D starts at +inf, so an exact tie implies a previous admissible pair.
__device__ __forceinline__ void consider(Best& b, bool adm, float D, int ju, int jd,
                                         const uint16_t* __restrict__ idx_up, const uint16_t* __restrict__ idx_dn) {
    bool better = adm && D < b.D;
    if (adm && D == b.D) better = tie_lower(idx_up, idx_dn, ju, jd, b.ju, b.jd);
    b.D = better ? D : b.D;
    b.ju = better ? ju : b.ju;
    b.jd = better ? jd : b.jd;
}

// The cells a window touches in one neighbour row, as ONE sequence of nt sorted positions: the first na start at a0
// (z bin zb0, strips ys0..ys1 are contiguous in the sorted row), the rest at b0 (z bin zb1 when the window crosses a
// bin edge).  Valid for zb1 - zb0 <= 1 (the default grid: bins wider than the window).
struct CellSeq {
    int a0, na, b0, nt;
};

__device__ __forceinline__ CellSeq window_cells(const DevGeom& g, const RowView& row, float ylo, float yhi, int zb0,
                                                int zb1) {
    const int ys0 = ybin(ylo, row.y0, row.inv_sy, g.ny), ys1 = ybin(yhi, row.y0, row.inv_sy, g.ny) + 1;
    const uint16_t* ta = row.tbl + zb0 * g.ny;
    CellSeq c;
    c.a0 = ta[ys0];
    c.na = (int)ta[ys1] - c.a0;
    c.b0 = 0;
    c.nt = c.na;
    if (zb1 > zb0) {
        const uint16_t* tb = row.tbl + zb1 * g.ny;
        c.b0 = tb[ys0];
        c.nt += (int)tb[ys1] - c.b0;
    }
    return c;
}

// Search window of one hit towards one neighbour row: pre-rounded bounds and the z bins they touch.
struct Win {
    float ylo, yhi, zlo, zhi;
    int zb0, zb1;
};

__device__ __forceinline__ Win make_win(const DevGeom& g, float y, float z, float wy, float wz, float z0) {
    Win w;
    w.ylo = __fsub_rn(y, wy);
    w.yhi = __fadd_rn(y, wy);
    w.zlo = __fsub_rn(z, wz);
    w.zhi = __fadd_rn(z, wz);
    w.zb0 = zbin(w.zlo, z0, g.inv_cz, g.nz);
    w.zb1 = zbin(w.zhi, z0, g.inv_cz, g.nz);
    return w;
}

// Exact search without the register lists (more than kNbList window hits in a neighbour row, or a grid finer than the
// window).  wu / wd: weights of the two first differences (reading A5'; 1 on equally spaced rows).
__device__ __noinline__ void search_dense(const DevGeom& g, const RowView& up, const RowView& dn, float y, float z,
                                          const Win& U, const Win& W, float wu, float wd, Best& best) {
    const int us0 = ybin(U.ylo, up.y0, up.inv_sy, g.ny), us1 = ybin(U.yhi, up.y0, up.inv_sy, g.ny);
    const int ds0 = ybin(W.ylo, dn.y0, dn.inv_sy, g.ny), ds1 = ybin(W.yhi, dn.y0, dn.inv_sy, g.ny);
    for (int zu = U.zb0; zu <= U.zb1; zu++) {
        const int u0 = up.tbl[zu * g.ny + us0], u1 = up.tbl[zu * g.ny + us1 + 1];
        for (int a = u0; a < u1; a++) {
            const float2 u = up.yz[a];
            if (!(U.ylo <= u.x && u.x <= U.yhi && U.zlo <= u.y && u.y <= U.zhi)) continue;
            const float a1 = __fmul_rn(wu, __fsub_rn(u.x, y)), a3 = __fmul_rn(wu, __fsub_rn(u.y, z));
            for (int zd = W.zb0; zd <= W.zb1; zd++) {
                const int d0 = dn.tbl[zd * g.ny + ds0], d1 = dn.tbl[zd * g.ny + ds1 + 1];
                for (int b = d0; b < d1; b++) {
                    const float2 d = dn.yz[b];
                    if (!(W.ylo <= d.x && d.x <= W.yhi && W.zlo <= d.y && d.y <= W.zhi)) continue;
                    const float ey = __fsub_rn(a1, __fmul_rn(wd, __fsub_rn(y, d.x)));
                    const float ez = __fsub_rn(a3, __fmul_rn(wd, __fsub_rn(z, d.y)));
                    const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));
                    consider(best, D <= g.nf_d2max, D, a, b, up.idx, dn.idx);
                }
            }
        }
    }
}

// ---- class 1 (reading A2', nf_bridge_rows = 1): a hit WITHOUT an admissible adjacent pair may take one partner two
// rows away, so that a single missing row does not break the chain.  (du, dd) = (1, 2): u in row r+1, d in row r-2;
// (2, 1): u in row r+2, d in row r-1.  The partner two rows away is searched in the doubled window; the deviation is
// dd * (u - h) - du * (h - d), i.e. (t1 + t1) - t2 resp. t1 - (t2 + t2); cut at 2.25 * d2max; minimum over
// (D, du, local index of u, local index of d).  Exact evaluation order: DESIGN.md "S2 class 1".  Rare (hits next to
// a missing cluster, and noise), so it is a plain out-of-line nested search over the grid cells.
struct BestBridge {
    float D;
    int ju, jd, du;  // positions in the sorted rows r+du / r-(3-du); ju < 0 = none
};

// Minimum over (D, du, local index of u, local index of d) for class 1, straight-line; b.D starts at +inf, b.du at 1,
// the (1,2) pairs are all considered before the (2,1) pairs, so a (2,1) pair never replaces a (1,2) pair on a tie.
__device__ __forceinline__ void consider_bridge(BestBridge& b, bool adm, float D, int du, int ju, int jd,
                                                const uint16_t* __restrict__ idx_up,
                                                const uint16_t* __restrict__ idx_dn) {
    bool better = adm && D < b.D;
    if (adm && D == b.D && du == b.du) better = tie_lower(idx_up, idx_dn, ju, jd, b.ju, b.jd);
    b.D = better ? D : b.D;
    b.ju = better ? ju : b.ju;
    b.jd = better ? jd : b.jd;
    b.du = better ? du : b.du;
}

template <bool kFarIsUp>
__device__ __forceinline__ void bridge_pairs(const DevGeom& g, const RowView& nearr, const RowView& farr, float y, float z,
                                             float z0, BestBridge& best) {
    const float WY = g.nf_wy, WZ = g.nf_wz, WY2 = __fadd_rn(WY, WY), WZ2 = __fadd_rn(WZ, WZ);
    const float dmax = __fmul_rn(g.nf_d2max, 2.25f);
    const float ylo = __fsub_rn(y, WY), yhi = __fadd_rn(y, WY), zlo = __fsub_rn(z, WZ), zhi = __fadd_rn(z, WZ);
    const float ylo2 = __fsub_rn(y, WY2), yhi2 = __fadd_rn(y, WY2), zlo2 = __fsub_rn(z, WZ2), zhi2 = __fadd_rn(z, WZ2);
    const int nz0 = zbin(zlo, z0, g.inv_cz, g.nz), nz1 = zbin(zhi, z0, g.inv_cz, g.nz);
    const int fz0 = zbin(zlo2, z0, g.inv_cz, g.nz), fz1 = zbin(zhi2, z0, g.inv_cz, g.nz);
    const int ns0 = ybin(ylo, nearr.y0, nearr.inv_sy, g.ny), ns1 = ybin(yhi, nearr.y0, nearr.inv_sy, g.ny);
    const int fs0 = ybin(ylo2, farr.y0, farr.inv_sy, g.ny), fs1 = ybin(yhi2, farr.y0, farr.inv_sy, g.ny);
    const int du = kFarIsUp ? 2 : 1;
    for (int zn = nz0; zn <= nz1; zn++) {
        const int a0 = nearr.tbl[zn * g.ny + ns0], a1 = nearr.tbl[zn * g.ny + ns1 + 1];
        for (int a = a0; a < a1; a++) {
            const float2 p = nearr.yz[a];
            if (!(ylo <= p.x && p.x <= yhi && zlo <= p.y && p.y <= zhi)) continue;
            for (int zf = fz0; zf <= fz1; zf++) {
                const int b0 = farr.tbl[zf * g.ny + fs0], b1 = farr.tbl[zf * g.ny + fs1 + 1];
                for (int b = b0; b < b1; b++) {
                    const float2 q = farr.yz[b];
                    if (!(ylo2 <= q.x && q.x <= yhi2 && zlo2 <= q.y && q.y <= zhi2)) continue;
                    // u = the upper partner, d = the lower one
                    const float2 u = kFarIsUp ? q : p, d = kFarIsUp ? p : q;
                    const int ju = kFarIsUp ? b : a, jd = kFarIsUp ? a : b;
                    const float t1 = __fsub_rn(u.x, y), t2 = __fsub_rn(y, d.x);
                    const float t3 = __fsub_rn(u.y, z), t4 = __fsub_rn(z, d.y);
                    const float ey = kFarIsUp ? __fsub_rn(t1, __fadd_rn(t2, t2)) : __fsub_rn(__fadd_rn(t1, t1), t2);
                    const float ez = kFarIsUp ? __fsub_rn(t3, __fadd_rn(t4, t4)) : __fsub_rn(__fadd_rn(t3, t3), t4);
                    const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));
                    if (!(D <= dmax)) continue;
                    bool better = best.ju < 0 || D < best.D;
                    if (!better && D == best.D && du == best.du) {  // (1,2) beats (2,1) on a tie; same kind: indices
                        const uint16_t* iu = kFarIsUp ? farr.idx : nearr.idx;
                        const uint16_t* id = kFarIsUp ? nearr.idx : farr.idx;
                        const int cu = iu[ju], bu = iu[best.ju];
                        better = cu < bu || (cu == bu && id[jd] < id[best.jd]);
                    }
                    if (better) {
                        best.D = D;
                        best.ju = ju;
                        best.jd = jd;
                        best.du = du;
                    }
                }
            }
        }
    }
}

__device__ __noinline__ void search_bridge(const DevGeom& g, const RowView& up, const RowView& dn, const RowView& up2,
                                           const RowView& dn2, bool has_up2, bool has_dn2, float y, float z, float z0,
                                           BestBridge& best) {
    if (has_dn2) bridge_pairs<false>(g, up, dn2, y, z, z0, best);  // (du, dd) = (1, 2) first: it wins exact ties
    if (has_up2) bridge_pairs<true>(g, dn, up2, y, z, z0, best);   // (du, dd) = (2, 1)
}

__device__ __forceinline__ bool in_window(float2 h, float ylo, float yhi, float zlo, float zhi) {
    return ylo <= h.x && h.x <= yhi && zlo <= h.y && h.y <= zhi;
}


// Window hits of one adjacent row as a register list: (first coordinate difference, second) of the newest four,
// their sorted positions (newest in the low 16 bits), and how many there are.
struct NearList {
    float pa, pb, pc, pd, qa, qb, qc, qd;
    unsigned long long pos;
    int n;
};

// kUp: the list holds (y_u - y, z_u - z) of row r+1; else (y - y_d, z - z_d) of row r-1.
template <bool kUp>
__device__ __forceinline__ NearList near_list(const DevGeom& g, const RowView& row, float y, float z, float ylo,
                                              float yhi, float zlo, float zhi, int zb0, int zb1) {
    const CellSeq c = window_cells(g, row, ylo, yhi, zb0, zb1);
    const int shift = c.b0 - c.na;
    NearList l{0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0.0f, 0ull, 0};
    for (int k = 0; k < c.nt; k++) {
        const int j = k < c.na ? c.a0 + k : k + shift;
        const float2 h = row.yz[j];
        const bool in = in_window(h, ylo, yhi, zlo, zhi);
        const float p = kUp ? __fsub_rn(h.x, y) : __fsub_rn(y, h.x), q = kUp ? __fsub_rn(h.y, z) : __fsub_rn(z, h.y);
        l.pd = in ? l.pc : l.pd; l.pc = in ? l.pb : l.pc; l.pb = in ? l.pa : l.pb; l.pa = in ? p : l.pa;
        l.qd = in ? l.qc : l.qd; l.qc = in ? l.qb : l.qc; l.qb = in ? l.qa : l.qb; l.qa = in ? q : l.qa;
        l.pos = in ? ((l.pos << 16) | (unsigned long long)j) : l.pos;
        l.n += in ? 1 : 0;
    }
    return l;
}

// The cells of the doubled window in a row two away, as one sequence of up to three contiguous ranges.
struct FarSeq {
    int s0, n0, s1, n1, s2, nt;
};

__device__ __forceinline__ FarSeq far_cells(const DevGeom& g, const RowView& row, float ylo2, float yhi2, int fz0,
                                            int fz1) {
    const int fs0 = ybin(ylo2, row.y0, row.inv_sy, g.ny), fs1 = ybin(yhi2, row.y0, row.inv_sy, g.ny) + 1;
    FarSeq f{0, 0, 0, 0, 0, 0};
    f.s0 = row.tbl[fz0 * g.ny + fs0];
    f.n0 = (int)row.tbl[fz0 * g.ny + fs1] - f.s0;
    f.nt = f.n0;
    if (fz1 > fz0) {
        f.s1 = row.tbl[(fz0 + 1) * g.ny + fs0];
        f.n1 = (int)row.tbl[(fz0 + 1) * g.ny + fs1] - f.s1;
        f.nt += f.n1;
    }
    if (fz1 > fz0 + 1) {
        f.s2 = row.tbl[(fz0 + 2) * g.ny + fs0];
        f.nt += (int)row.tbl[(fz0 + 2) * g.ny + fs1] - f.s2;
    }
    return f;
}

__device__ __forceinline__ int far_pos(const FarSeq& f, int k) {
    return k < f.n0 ? f.s0 + k : (k < f.n0 + f.n1 ? f.s1 + (k - f.n0) : f.s2 + (k - f.n0 - f.n1));
}

#ifndef TPC_NB_FAR
#define TPC_NB_FAR 1
#endif
#ifndef TPC_BR_CTAS
#define TPC_BR_CTAS 8
#endif
constexpr int kNbFar = TPC_NB_FAR;  // hits of a row two away fetched together before they are examined

// Class-1 search of one hit (see above search_bridge for the reading).  Flat loops over the cells of the rows two
// away, paired with the register lists of the adjacent rows; dense spots and fine grids take the nested search.
__device__ __forceinline__ BestBridge bridge_hit(const DevGeom& g, const RowView& up, const RowView& dn,
                                                 const RowView& up2, const RowView& dn2, bool has_up2, bool has_dn2,
                                                 float y, float z, float z0) {
    const float WY = g.nf_wy, WZ = g.nf_wz;
    const float kInf = __int_as_float(0x7f800000);
    BestBridge bb{kInf, -1, -1, 1};
    const float ylo = __fsub_rn(y, WY), yhi = __fadd_rn(y, WY), zlo = __fsub_rn(z, WZ), zhi = __fadd_rn(z, WZ);
    const int zb0 = zbin(zlo, z0, g.inv_cz, g.nz), zb1 = zbin(zhi, z0, g.inv_cz, g.nz);
    const float WY2 = __fadd_rn(WY, WY), WZ2 = __fadd_rn(WZ, WZ), dmax = __fmul_rn(g.nf_d2max, 2.25f);
    const float ylo2 = __fsub_rn(y, WY2), yhi2 = __fadd_rn(y, WY2), zlo2 = __fsub_rn(z, WZ2), zhi2 = __fadd_rn(z, WZ2);
    const int fz0 = zbin(zlo2, z0, g.inv_cz, g.nz), fz1 = zbin(zhi2, z0, g.inv_cz, g.nz);
    bool generic = zb1 - zb0 > 1 || fz1 - fz0 > 2;
    if (!generic) {
        const NearList lu = near_list<true>(g, up, y, z, ylo, yhi, zlo, zhi, zb0, zb1);
        const NearList ld = near_list<false>(g, dn, y, z, ylo, yhi, zlo, zhi, zb0, zb1);
        generic = lu.n > kNbList || ld.n > kNbList;
        if (!generic && lu.n > 0 && has_dn2) {  // (du, dd) = (1, 2): u from the row r+1 list, d in row r-2
            const FarSeq f = far_cells(g, dn2, ylo2, yhi2, fz0, fz1);
            float2 fh[kNbFar];  // the first far hits are loaded together (one memory round trip), then examined
#pragma unroll
            for (int k = 0; k < kNbFar; k++) fh[k] = k < f.nt ? dn2.yz[far_pos(f, k)] : make_float2(0.0f, 0.0f);
#pragma unroll 1
            for (int k = 0; k < f.nt; k++) {
                const int b = far_pos(f, k);
                float2 d;
                if (k < kNbFar) {
                    d = fh[0];
#pragma unroll
                    for (int q = 0; q < kNbFar - 1; q++) fh[q] = fh[q + 1];  // shift: no dynamic register indexing
                } else {
                    d = dn2.yz[b];
                }
                const bool din = in_window(d, ylo2, yhi2, zlo2, zhi2);
                if (!din) continue;  // the cells cover several times the window: most far hits end here
                const float t2 = __fsub_rn(y, d.x), t4 = __fsub_rn(z, d.y);
#define TPC_NB_BRIDGE_A(T1, T3, Q)                                                                             \
    {                                                                                                          \
        const float ey = __fsub_rn(__fadd_rn(T1, T1), t2), ez = __fsub_rn(__fadd_rn(T3, T3), t4);              \
        const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));                                       \
        consider_bridge(bb, din && lu.n > Q && D <= dmax, D, 1, (int)((lu.pos >> (16 * Q)) & 0xffffull), b, up.idx, \
                        dn2.idx);                                                                              \
    }
                TPC_NB_BRIDGE_A(lu.pa, lu.qa, 0)
                if (lu.n > 1) {
                    TPC_NB_BRIDGE_A(lu.pb, lu.qb, 1)
                    TPC_NB_BRIDGE_A(lu.pc, lu.qc, 2)
                    TPC_NB_BRIDGE_A(lu.pd, lu.qd, 3)
                }
#undef TPC_NB_BRIDGE_A
            }
        }
        if (!generic && ld.n > 0 && has_up2) {  // (du, dd) = (2, 1): u in row r+2, d from the row r-1 list
            const FarSeq f = far_cells(g, up2, ylo2, yhi2, fz0, fz1);
            float2 fh[kNbFar];
#pragma unroll
            for (int k = 0; k < kNbFar; k++) fh[k] = k < f.nt ? up2.yz[far_pos(f, k)] : make_float2(0.0f, 0.0f);
#pragma unroll 1
            for (int k = 0; k < f.nt; k++) {
                const int a = far_pos(f, k);
                float2 u;
                if (k < kNbFar) {
                    u = fh[0];
#pragma unroll
                    for (int q = 0; q < kNbFar - 1; q++) fh[q] = fh[q + 1];
                } else {
                    u = up2.yz[a];
                }
                const bool uin = in_window(u, ylo2, yhi2, zlo2, zhi2);
                if (!uin) continue;
                const float t1 = __fsub_rn(u.x, y), t3 = __fsub_rn(u.y, z);
#define TPC_NB_BRIDGE_B(T2, T4, Q)                                                                             \
    {                                                                                                          \
        const float ey = __fsub_rn(t1, __fadd_rn(T2, T2)), ez = __fsub_rn(t3, __fadd_rn(T4, T4));              \
        const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));                                       \
        consider_bridge(bb, uin && ld.n > Q && D <= dmax, D, 2, a, (int)((ld.pos >> (16 * Q)) & 0xffffull), up2.idx, \
                        dn.idx);                                                                               \
    }
                TPC_NB_BRIDGE_B(ld.pa, ld.qa, 0)
                if (ld.n > 1) {
                    TPC_NB_BRIDGE_B(ld.pb, ld.qb, 1)
                    TPC_NB_BRIDGE_B(ld.pc, ld.qc, 2)
                    TPC_NB_BRIDGE_B(ld.pd, ld.qd, 3)
                }
#undef TPC_NB_BRIDGE_B
            }
        }
    }
    if (generic) {
        bb = BestBridge{kInf, -1, -1, 1};
        search_bridge(g, up, dn, up2, dn2, has_up2, has_dn2, y, z, z0, bb);
    }
    return bb;
}

// r = pad row of the hits (1..R-2).  Reading A5': the window towards row r+1 / r-1 has half-sizes (WY, WZ) * su / sd
// and the deviation is wu (u - h) - wd (h - d); all four factors are exactly 1 on equally spaced rows, where this is
// the plain second difference of the default reading (x * 1.0f is exact).
// kUniform: all rows equally spaced -- the factors are all 1, so the multiplications and the second window are
// skipped (same bits: x * 1.0f is exact); the launcher picks the variant from the geometry.
template <bool kUniform>
__device__ __forceinline__ float wmul(float w, float x) { return kUniform ? x : __fmul_rn(w, x); }

template <bool kUniform>
__device__ __forceinline__ void search_row(const DevGeom& g, const RowView up, const RowView dn, const float2* my_yz,
                                           int n, int r, float z0, int base, int base_up, int base_dn,
                                           int32_t* __restrict__ link_up, int32_t* __restrict__ link_dn) {
    const float D2MAX = g.nf_d2max;
    const float wu = kUniform ? 1.0f : g.row_wu[r], wd = kUniform ? 1.0f : g.row_wd[r];
    const float WYu = kUniform ? g.nf_wy : __fmul_rn(g.nf_wy, g.row_su[r]);
    const float WZu = kUniform ? g.nf_wz : __fmul_rn(g.nf_wz, g.row_su[r]);
    const float WYd = kUniform ? g.nf_wy : __fmul_rn(g.nf_wy, g.row_sd[r]);
    const float WZd = kUniform ? g.nf_wz : __fmul_rn(g.nf_wz, g.row_sd[r]);
    const float kInf = __int_as_float(0x7f800000);
    for (int i = threadIdx.x; i < n; i += kNbThreads) {
        const float2 h = my_yz[i];
        const float y = h.x, z = h.y;
        const Win U = make_win(g, y, z, WYu, WZu, z0);
        const Win W = kUniform ? U : make_win(g, y, z, WYd, WZd, z0);
        Best best{kInf, -1, -1};
        // row r-1 window hits (the newest kNbList = 4) as wd * (y - y_d), wd * (z - z_d) plus their positions
        float t2a = 0.0f, t2b = 0.0f, t2c = 0.0f, t2d = 0.0f, t4a = 0.0f, t4b = 0.0f, t4c = 0.0f, t4d = 0.0f;
        unsigned long long ld = 0ull;
        int nd = 0;
        const bool coarse = U.zb1 - U.zb0 <= 1 && W.zb1 - W.zb0 <= 1;
        if (!coarse) {  // a grid finer than the window (non-default grid_cell_z): generic exact search
            search_dense(g, up, dn, y, z, U, W, wu, wd, best);
        } else {
            // Flat loops over the handful of hits in the touched cells.  Row r-1 first: its window hits (the newest
            // kNbList = 4) stay in registers plus their positions; then every window hit of row r+1 is paired with
            // them.  All straight-line code with predicates: the lanes of a warp see different hit counts, and
            // branches taken by a few lanes cost the whole warp.
            const CellSeq cd = window_cells(g, dn, W.ylo, W.yhi, W.zb0, W.zb1);
            const CellSeq cu = window_cells(g, up, U.ylo, U.yhi, U.zb0, U.zb1);
            const int dshift = cd.b0 - cd.na, ushift = cu.b0 - cu.na;
            for (int k = 0; k < cd.nt; k++) {
                const int j = k < cd.na ? cd.a0 + k : k + dshift;
                const float2 d = dn.yz[j];
                const bool in = in_window(d, W.ylo, W.yhi, W.zlo, W.zhi);
                const float a2 = wmul<kUniform>(wd, __fsub_rn(y, d.x)), a4 = wmul<kUniform>(wd, __fsub_rn(z, d.y));
                t2d = in ? t2c : t2d; t2c = in ? t2b : t2c; t2b = in ? t2a : t2b; t2a = in ? a2 : t2a;
                t4d = in ? t4c : t4d; t4c = in ? t4b : t4c; t4b = in ? t4a : t4b; t4a = in ? a4 : t4a;
                ld = in ? ((ld << 16) | (unsigned long long)j) : ld;
                nd += in ? 1 : 0;
            }
            if (nd <= kNbList) {
                bool tie = false;
                for (int k = 0; k < (nd > 0 ? cu.nt : 0); k++) {
                    const int ja = k < cu.na ? cu.a0 + k : k + ushift;
                    const float2 u = up.yz[ja];
                    const bool uin = in_window(u, U.ylo, U.yhi, U.zlo, U.zhi);
                    const float t1 = wmul<kUniform>(wu, __fsub_rn(u.x, y)), t3 = wmul<kUniform>(wu, __fsub_rn(u.y, z));
// strict minimum in visiting order; an exact tie of D with the best so far is only flagged (duplicated clusters, or
// perfectly straight synthetic tracks): such a hit is searched again by the exact out-of-line path below, so the
// common case pays no index comparison
#define TPC_NB_PAIR(T2, T4, Q)                                                                                   \
    {                                                                                                            \
        const float ey = __fsub_rn(t1, T2), ez = __fsub_rn(t3, T4);                                              \
        const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));                                         \
        const bool adm = uin && nd > Q && D <= D2MAX;                                                            \
        const bool lt = adm && D < best.D;                                                                       \
        tie = tie || (adm && D == best.D);                                                                       \
        best.D = lt ? D : best.D;                                                                                \
        best.ju = lt ? ja : best.ju;                                                                             \
        best.jd = lt ? (int)((ld >> (16 * Q)) & 0xffffull) : best.jd;                                            \
    }
                    TPC_NB_PAIR(t2a, t4a, 0)
                    TPC_NB_PAIR(t2b, t4b, 1)
                    if (nd > 2) {
                        TPC_NB_PAIR(t2c, t4c, 2)
                        TPC_NB_PAIR(t2d, t4d, 3)
                    }
#undef TPC_NB_PAIR
                }
                if (tie) {  // resolve by (D, local index of u, local index of d) exactly
                    best = Best{kInf, -1, -1};
                    search_dense(g, up, dn, y, z, U, W, wu, wd, best);
                }
            } else {
                // more than kNbList window hits in row r-1 (dense spots): pair every window hit of row r+1 with a
                // second pass over the row r-1 cells
                for (int k = 0; k < cu.nt; k++) {
                    const int ja = k < cu.na ? cu.a0 + k : k + ushift;
                    const float2 u = up.yz[ja];
                    if (!in_window(u, U.ylo, U.yhi, U.zlo, U.zhi)) continue;
                    const float t1 = wmul<kUniform>(wu, __fsub_rn(u.x, y)), t3 = wmul<kUniform>(wu, __fsub_rn(u.y, z));
                    for (int q = 0; q < cd.nt; q++) {
                        const int jb = q < cd.na ? cd.a0 + q : q + dshift;
                        const float2 d = dn.yz[jb];
                        const float ey = __fsub_rn(t1, wmul<kUniform>(wd, __fsub_rn(y, d.x)));
                        const float ez = __fsub_rn(t3, wmul<kUniform>(wd, __fsub_rn(z, d.y)));
                        const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));
                        consider(best, in_window(d, W.ylo, W.yhi, W.zlo, W.zhi) && D <= D2MAX, D, ja, jb, up.idx, dn.idx);
                    }
                }
            }
        }
        // links live in SORTED space: entry base + i belongs to the i-th hit of the sorted row, values are sorted
        // global positions; coalesced stores
        int lu = best.ju < 0 ? -1 : base_up + best.ju;
        int ldn = best.jd < 0 ? -1 : base_dn + best.jd;
        link_up[base + i] = lu;
        link_dn[base + i] = ldn;
    }
}

// ---- bulk copies into shared memory (TMA, 1-D) completing on an mbarrier ----
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "NB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra NB_DONE;\n"
        "bra NB_WAIT;\n"
        "NB_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

// global -> shared, src and dst 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// One CTA per (sector instance, pad row) slab.  The cell tables and the sorted hits of the rows r-1, r and r+1 come
// into shared memory by 1-D bulk copies (TMA) that one thread issues, all completing on one mbarrier: nobody spends
// instructions on staging (15 % of the kernel's instructions when every thread copied its share), and the copies of
// one CTA overlap the search of the others on the SM.  Rows longer than the buffer (cap_hits) and tables beyond
// kNbStageTbl entries are read in place.  (A CTA walking a segment of 2..16 consecutive rows through a ring of
// buffers, each row fetched once instead of three times, was measured too: 4.11-4.51 ms against 4.09 ms -- the
// per-row barrier costs more than the L2 reads it saves.)
#ifndef TPC_NB_CTAS
#define TPC_NB_CTAS 12  // resident CTAs per SM the register allocation aims at; measured 8 -> 4.09, 10 -> 3.90, 12 -> 3.87, 13 -> 3.97 ms
#endif
struct NbSmem {
    int tbl_bytes;  // bytes of one staged cell table (0 = tables are read in place)
    int cap_hits;   // hits of a row that fit its buffer
    int buf_bytes;  // buffer of a neighbour row: table, then (cap_hits + 2) hits (a copy may start 8 bytes before the row)
    int own_bytes;  // buffer of the own row: hits only
};
// buffers in shared memory: row r-1 | row r (hits only) | row r+1
__device__ __forceinline__ unsigned char* nb_buf(unsigned char* base, const NbSmem& sm, int k) {
    return base + (k == 0 ? 0 : (k == 1 ? sm.buf_bytes : sm.buf_bytes + sm.own_bytes));
}

template <bool kUniform>
__global__ void __launch_bounds__(kNbThreads, TPC_NB_CTAS)
neighbours_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
                  const float2* __restrict__ hit_yz, const uint16_t* __restrict__ hit_idx,
                  const uint16_t* __restrict__ bin_start, int32_t* __restrict__ link_up,
                  int32_t* __restrict__ link_dn, const NbSmem sm) {
    extern __shared__ __align__(128) unsigned char sm_raw[];
    __shared__ __align__(8) unsigned long long s_bar;
    const int slab = blockIdx.x;
    const int inst = slab / g.R, r = slab - inst * g.R;
    const int base = row_offsets[slab];
    const int n_all = row_offsets[slab + 1] - base;
    const int n = min(n_all, 65535);
    // hits beyond the 16-bit limit were not binned (error flag set by S1): they own no links
    for (int i = n + threadIdx.x; i < n_all; i += kNbThreads) link_up[base + i] = link_dn[base + i] = -1;
    if (r == 0 || r == g.R - 1) {  // first and last row never own links (reading A6)
        for (int i = threadIdx.x; i < n; i += kNbThreads) link_up[base + i] = link_dn[base + i] = -1;
        return;
    }
    if (n == 0) return;
    const int base_dn = row_offsets[slab - 1], base_up = row_offsets[slab + 1];
    const int n_dn = min(base - base_dn, 65535), n_up = min(row_offsets[slab + 2] - base_up, 65535);
    // row q = r - 1 + k (k = 0, 1, 2) lives in buffer k
    const int off3[3] = {base_dn, base, base_up};
    const int cnt3[3] = {n_dn, n, n_up};
    if (threadIdx.x == 0) {
        mbar_init(&s_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        unsigned bytes = 0;
        unsigned hb[3], lead[3];
#pragma unroll
        for (int k = 0; k < 3; k++) {
            lead[k] = (unsigned)((uintptr_t)(hit_yz + off3[k]) & 15u);  // 0 or 8: the copy starts at the 16-byte line
            hb[k] = (cnt3[k] > 0 && cnt3[k] <= sm.cap_hits) ? (((unsigned)cnt3[k] * 8u + lead[k] + 15u) & ~15u) : 0u;
            bytes += hb[k] + (k != 1 ? (unsigned)sm.tbl_bytes : 0u);  // the own row's table is not needed
        }
        mbar_expect_tx(&s_bar, bytes);
#pragma unroll
        for (int k = 0; k < 3; k++) {
            unsigned char* buf = nb_buf(sm_raw, sm, k);
            if (k != 1 && sm.tbl_bytes)
                bulk_g2s(buf, bin_start + (size_t)(slab - 1 + k) * g.nzp, (unsigned)sm.tbl_bytes, &s_bar);
            if (hb[k])
                bulk_g2s(buf + (k != 1 ? sm.tbl_bytes : 0), reinterpret_cast<const unsigned char*>(hit_yz + off3[k]) - lead[k], hb[k],
                         &s_bar);
        }
    }
    __syncthreads();  // the barrier is initialised before anybody waits on it
    const float z0 = grid_z0(g, inst);
    RowView v[3];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        unsigned char* buf = nb_buf(sm_raw, sm, k);
        const float2* src = hit_yz + off3[k];
        const unsigned lead = (unsigned)((uintptr_t)src & 15u);
        v[k].yz = (cnt3[k] <= sm.cap_hits) ? reinterpret_cast<const float2*>(buf + (k != 1 ? sm.tbl_bytes : 0) + lead) : src;
        v[k].idx = hit_idx + off3[k];
        v[k].tbl = sm.tbl_bytes ? reinterpret_cast<const uint16_t*>(buf) : bin_start + (size_t)(slab - 1 + k) * g.nzp;
        v[k].y0 = g.row_y0[r - 1 + k];
        v[k].inv_sy = g.row_inv_sy[r - 1 + k];
    }
    mbar_wait(&s_bar, 0u);
    search_row<kUniform>(g, v[2], v[0], v[1].yz, n, r, z0, base, base_up, base_dn, link_up, link_dn);
}

// Class 1 (reading A2', nf_bridge_rows = 1) as its own pass: one WARP per (instance,row) slab reads the row's raw
// up-links, queues the hits without an adjacent pair (about one in five) and searches 32 of them at a time, so the
// lanes stay busy and the tuned class-0 kernel above is untouched.  All rows are read in place (L2).
constexpr int kBrThreads = 128;

__global__ void __launch_bounds__(kBrThreads, TPC_BR_CTAS)
bridge_links_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
                    const float2* __restrict__ hit_yz, const uint16_t* __restrict__ hit_idx,
                    const uint16_t* __restrict__ bin_start, int32_t* __restrict__ link_up,
                    int32_t* __restrict__ link_dn, int n_slabs) {
    __shared__ uint16_t s_queue[kBrThreads / 32][64];
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int slab = blockIdx.x * (kBrThreads / 32) + wid;
    if (slab >= n_slabs) return;
    const int inst = slab / g.R, r = slab - inst * g.R;
    if (r == 0 || r == g.R - 1) return;  // first and last row never own links (reading A6)
    const int base = row_offsets[slab];
    const int n = min(row_offsets[slab + 1] - base, 65535);
    if (n == 0) return;
    const float z0 = grid_z0(g, inst);
    const bool has_up2 = r + 2 <= g.R - 1, has_dn2 = r - 2 >= 0;
    const int base_dn = row_offsets[slab - 1], base_up = row_offsets[slab + 1];
    const int base_up2 = has_up2 ? row_offsets[slab + 2] : 0, base_dn2 = has_dn2 ? row_offsets[slab - 2] : 0;
    const int ru2 = has_up2 ? r + 2 : r, rd2 = has_dn2 ? r - 2 : r;
    const RowView up{hit_yz + base_up, hit_idx + base_up, bin_start + (size_t)(slab + 1) * g.nzp, g.row_y0[r + 1],
                     g.row_inv_sy[r + 1]};
    const RowView dn{hit_yz + base_dn, hit_idx + base_dn, bin_start + (size_t)(slab - 1) * g.nzp, g.row_y0[r - 1],
                     g.row_inv_sy[r - 1]};
    const RowView up2{hit_yz + base_up2, hit_idx + base_up2, bin_start + (size_t)(slab + (has_up2 ? 2 : 0)) * g.nzp,
                      g.row_y0[ru2], g.row_inv_sy[ru2]};
    const RowView dn2{hit_yz + base_dn2, hit_idx + base_dn2, bin_start + (size_t)(slab - (has_dn2 ? 2 : 0)) * g.nzp,
                      g.row_y0[rd2], g.row_inv_sy[rd2]};
    uint16_t* queue = s_queue[wid];
    const unsigned lt = (1u << lane) - 1u;
    int qn = 0;  // queued hits (warp-uniform), < 32 between rounds
    for (int i0 = 0; i0 < n || qn > 0; i0 += 32) {
        const int i = i0 + lane;
        const bool need = i < n && link_up[base + i] < 0;
        const unsigned m = __ballot_sync(0xffffffffu, need);
        if (need) queue[qn + __popc(m & lt)] = (uint16_t)i;
        qn += __popc(m);
        __syncwarp();
        const bool last = i0 + 32 >= n;
        if (qn >= 32 || (last && qn > 0)) {
            const int take = min(qn, 32);
            if (lane < take) {
                const int j = queue[lane];
                const float2 h = hit_yz[base + j];
                const BestBridge bb = bridge_hit(g, up, dn, up2, dn2, has_up2, has_dn2, h.x, h.y, z0);
                if (bb.ju >= 0) {
                    link_up[base + j] = (bb.du == 2 ? base_up2 : base_up) + bb.ju;
                    link_dn[base + j] = (bb.du == 2 ? base_dn : base_dn2) + bb.jd;
                }
            }
            __syncwarp();
            const uint16_t moved = lane + 32 < qn ? queue[lane + 32] : (uint16_t)0;
            __syncwarp();
            if (lane + 32 < qn) queue[lane] = moved;
            qn -= take;
            __syncwarp();
        }
        if (last && qn == 0) break;
    }
}

static NbSmem nb_smem(const DevGeom& g) {
    NbSmem m;
    m.tbl_bytes = g.nzp <= kNbStageTbl ? g.nzp * 2 : 0;  // nzp is a multiple of 16 entries
    m.cap_hits = kNbStageHits;
    m.buf_bytes = (m.tbl_bytes + (m.cap_hits + 2) * 8 + 127) & ~127;
    m.own_bytes = ((m.cap_hits + 2) * 8 + 127) & ~127;
    return m;
}

int launch_neighbours(const DevGeom& g, const Workspace& w, const Problem& p, cudaStream_t s) {
    const int slabs = p.n_inst * g.R;
    if (slabs == 0) return 0;
    const NbSmem m = nb_smem(g);
    const size_t smem = (size_t)m.buf_bytes * 2 + m.own_bytes;
    if (g.uniform_pitch)
        neighbours_kernel<true><<<slabs, kNbThreads, smem, s>>>(g, p.row_offsets, w.hit_yz, w.hit_idx, w.bin_start,
                                                                w.up_raw, w.dn_raw, m);
    else
        neighbours_kernel<false><<<slabs, kNbThreads, smem, s>>>(g, p.row_offsets, w.hit_yz, w.hit_idx, w.bin_start,
                                                                 w.up_raw, w.dn_raw, m);
    if (g.bridge) {  // class 1 (reading A2'): a second, light pass over the hits that found no adjacent pair
        bridge_links_kernel<<<div_up(slabs, kBrThreads / 32), kBrThreads, 0, s>>>(g, p.row_offsets, w.hit_yz, w.hit_idx,
                                                                                  w.bin_start, w.up_raw, w.dn_raw, slabs);
        return 2;
    }
    return 1;
}

}  // namespace tpc
