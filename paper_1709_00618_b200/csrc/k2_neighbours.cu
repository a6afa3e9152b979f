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
// One CTA per (sector instance, pad row).  The sorted (y,z), the original indices and the bin tables of the two
// adjacent rows are staged in shared memory (they are read ~10x per hit); rows too long for that are read in place.
#include "tpc_common.cuh"

namespace tpc {

constexpr int kNbThreads = 128;
constexpr int kNbStageHits = 3584;  // max hits of row r-1 plus row r+1 staged in shared memory (10 B each)

struct RowView {
    const float2* yz;
    const uint16_t* idx;
    const uint16_t* tbl;
};

__device__ __forceinline__ void search_row(const DevGeom& g, const RowView up, const RowView dn, const float2* my_yz,
                                           const uint16_t* my_idx, int n, float z0, int base, int base_up,
                                           int base_dn, int32_t* __restrict__ link_up,
                                           int32_t* __restrict__ link_dn) {
    const float WY = g.nf_wy, WZ = g.nf_wz, D2MAX = g.nf_d2max;
    for (int i = threadIdx.x; i < n; i += kNbThreads) {
        const float2 h = my_yz[i];
        const float y = h.x, z = h.y;
        const float ylo = __fsub_rn(y, WY), yhi = __fadd_rn(y, WY);
        const float zlo = __fsub_rn(z, WZ), zhi = __fadd_rn(z, WZ);
        const int b0 = zbin(zlo, z0, g.inv_cz, g.nz), b1 = zbin(zhi, z0, g.inv_cz, g.nz);
        const int u0 = up.tbl[b0], u1 = up.tbl[b1 + 1];
        const int d0 = dn.tbl[b0], d1 = dn.tbl[b1 + 1];
        int bu = -1, bd = -1;
        float bD = 0.0f;
        for (int a = u0; a < u1; a++) {
            const float2 u = up.yz[a];
            if (!(ylo <= u.x && u.x <= yhi && zlo <= u.y && u.y <= zhi)) continue;
            const float t1 = __fsub_rn(u.x, y), t3 = __fsub_rn(u.y, z);
            const int iu = up.idx[a];
            for (int b = d0; b < d1; b++) {
                const float2 d = dn.yz[b];
                if (!(ylo <= d.x && d.x <= yhi && zlo <= d.y && d.y <= zhi)) continue;
                const float t2 = __fsub_rn(y, d.x), ey = __fsub_rn(t1, t2);
                const float t4 = __fsub_rn(z, d.y), ez = __fsub_rn(t3, t4);
                const float D = __fadd_rn(__fmul_rn(ey, ey), __fmul_rn(ez, ez));
                if (!(D <= D2MAX)) continue;
                bool better = bu < 0 || D < bD;
                if (!better && D == bD) {
                    const int id = dn.idx[b];
                    better = iu < bu || (iu == bu && id < bd);
                }
                if (better) {
                    bD = D;
                    bu = iu;
                    bd = dn.idx[b];
                }
            }
        }
        const int me = base + my_idx[i];
        link_up[me] = bu < 0 ? -1 : base_up + bu;
        link_dn[me] = bd < 0 ? -1 : base_dn + bd;
    }
}

__global__ void __launch_bounds__(kNbThreads)
neighbours_kernel(const __grid_constant__ DevGeom g, const int32_t* __restrict__ row_offsets,
                  const float2* __restrict__ hit_yz, const uint16_t* __restrict__ hit_idx,
                  const uint16_t* __restrict__ bin_start, int32_t* __restrict__ link_up,
                  int32_t* __restrict__ link_dn) {
    extern __shared__ __align__(16) unsigned char sm_raw[];
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
    const int base_dn = row_offsets[slab - 1], base_up = row_offsets[slab + 1];
    const int n_dn = min(base - base_dn, 65535), n_up = min(row_offsets[slab + 2] - base_up, 65535);
    const float z0 = grid_z0(g, inst);
    const uint16_t* tbl_up = bin_start + (size_t)(slab + 1) * g.nzp;
    const uint16_t* tbl_dn = bin_start + (size_t)(slab - 1) * g.nzp;
    RowView up, dn;
    if (n_up + n_dn <= kNbStageHits) {
        // shared layout: yz_up[n_up] yz_dn[n_dn] | tbl_up[nzp] tbl_dn[nzp] idx_up[n_up] idx_dn[n_dn]
        float2* s_yz = reinterpret_cast<float2*>(sm_raw);
        uint16_t* s_16 = reinterpret_cast<uint16_t*>(s_yz + kNbStageHits);
        uint16_t* s_tu = s_16;
        uint16_t* s_td = s_16 + g.nzp;
        uint16_t* s_iu = s_td + g.nzp;
        uint16_t* s_id = s_iu + n_up;
        for (int i = threadIdx.x; i < n_up; i += kNbThreads) {
            s_yz[i] = __ldg(&hit_yz[base_up + i]);
            s_iu[i] = __ldg(&hit_idx[base_up + i]);
        }
        for (int i = threadIdx.x; i < n_dn; i += kNbThreads) {
            s_yz[n_up + i] = __ldg(&hit_yz[base_dn + i]);
            s_id[i] = __ldg(&hit_idx[base_dn + i]);
        }
        for (int i = threadIdx.x; i <= g.nz; i += kNbThreads) {
            s_tu[i] = __ldg(&tbl_up[i]);
            s_td[i] = __ldg(&tbl_dn[i]);
        }
        __syncthreads();
        up = RowView{s_yz, s_iu, s_tu};
        dn = RowView{s_yz + n_up, s_id, s_td};
    } else {
        up = RowView{hit_yz + base_up, hit_idx + base_up, tbl_up};
        dn = RowView{hit_yz + base_dn, hit_idx + base_dn, tbl_dn};
    }
    search_row(g, up, dn, hit_yz + base, hit_idx + base, n, z0, base, base_up, base_dn, link_up, link_dn);
}

static size_t nb_smem_bytes(const DevGeom& g) {
    return (size_t)kNbStageHits * sizeof(float2) + (size_t)(2 * g.nzp + kNbStageHits) * sizeof(uint16_t);
}

int launch_neighbours(const DevGeom& g, const Workspace& w, const Problem& p, cudaStream_t s) {
    const int slabs = p.n_inst * g.R;
    if (slabs == 0) return 0;
    static bool configured = false;
    const size_t smem = nb_smem_bytes(g);
    if (!configured) {
        cudaFuncSetAttribute(neighbours_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
        configured = true;
    }
    neighbours_kernel<<<slabs, kNbThreads, smem, s>>>(g, p.row_offsets, w.hit_yz, w.hit_idx, w.bin_start, w.up_raw,
                                                      w.dn_raw);
    return 1;
}

}  // namespace tpc
