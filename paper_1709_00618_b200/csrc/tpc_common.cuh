// Internal declarations shared by the CUDA translation units of libtpctrk.so.  Not part of the ABI.
// (The CPU oracle in oracle/ includes nothing from here.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tpc {

constexpr int kCandMax = 10;      // TPC_CAND_MAX_HITS
constexpr int kMaxRows = 255;
constexpr size_t kVtxMaxSmemBytes = 200 * 1024;  // vertex_seeds_kernel keeps one window's z_v histogram in shared memory
constexpr int kMaxDeviceOrdinals = 64;  // per-device caches of kernel attributes (launch helpers)
constexpr int kMaxCells = 16384;  // cells of one row's grid (positions and the table are 16 bit; S1 keeps 4 B/cell in smem)
constexpr uint16_t kNoHit = 0xFFFFu;
constexpr float kKappaPerTesla = 0.00299792458f;

// Everything the kernels need to know about geometry and tunables.  Passed by value as a
// __grid_constant__ kernel parameter (lives in the constant bank; uniform reads are free).
struct DevGeom {
    int R;          // pad rows
    int RP;         // row stride of the per-tracklet hit table (R rounded up to 8)
    int sel_words;  // 32-bit words of a tracklet's kept-row mask (S6): ceil(R / 32)
    int sel_stride; // words per S6 tracklet record: mask, track index, first hit position; multiple of 4 (16 B)
    int nz;         // z bins per row
    int ny;         // y strips per row
    int ncell;      // nz * ny cells per row, cell id = zbin * ny + ystrip (a y range inside one z bin is contiguous)
    int nzp;        // stride of the cell table (ncell + 1 rounded up to 16 entries = 32 B)
    int spe, spe_half;
    int inst_phase;  // geometric sector of instance 0 of this call (0 except for the chunks of the host pipeline)
    float z0_a, z0_c;  // grid origin: z >= 0 side, z < 0 side
    float inv_cz;
    float nf_wy, nf_wz, nf_d2max;
    int bridge;     // S2: 1 = a single missing row may be bridged (reading A2')
    int cand_min, cand_max;
    float p0[5];
    float gate, wmax;
    int max_gap;
    float max_s, edge_margin, tan_half;
    int sel_min;
    float cos_2h, sin_2h;  // rotation between neighbouring sector frames: angle 2 * half_angle
    int vtx_nb;            // bins of the per-window z_v histogram (0.5 cm over [-vtx_h, vtx_h))
    float vtx_h;
    float sy2, sz2;
    float cB;       // curvature per (q/pt): kappa = cB * q/pt
    const float* row_x;  // device [R]
    const float* row_y0;      // device [R] lower edge of the row's y grid: -(row half-width + 0.5 cm)
    const float* row_inv_sy;  // device [R] strips per cm of that row
    // S2 with a non-uniform row pitch (reading A5'): weights of the two first differences and scale of the search
    // window towards row r+1 / r-1; all exactly 1 on equally spaced rows
    int uniform_pitch;        // 1: every step factor below is exactly 1 (the S2 kernel skips them)
    const float* row_wu;      // device [R]
    const float* row_wd;
    const float* row_su;
    const float* row_sd;
};

// Views into the caller's workspace (all device pointers), fixed per call.
struct Workspace {
    float2* hit_yz;       // [N]  (y, z) sorted by grid cell inside every (instance,row) segment
    uint16_t* hit_idx;    // [N]  local index (position in the row segment of the INPUT) of the sorted hit
    uint16_t* hit_pos;    // [N]  inverse of hit_idx: position in the sorted row of the hit with that local index
    uint16_t* bin_start;  // [S*R][nzp] first sorted position of every grid cell, entry ncell = row length
    // Index spaces: everything below that is indexed by hit or holds hit indices uses SORTED global positions
    // (row start + position in the sorted row); the user-facing outputs are translated back through hit_idx.
    int32_t* up_raw;      // [N] S2 links
    int32_t* dn_raw;
    int32_t* up;          // [N] cleaned up-links (S3; the cleaned down-links are never materialised)
    uint32_t* claim;      // [N] S6 best claiming weight
    uint8_t* flags;       // [N] bit0 start hit, bit1 candidate
    int2* scan_tmp;       // [S*R / 4096 + 2] tile totals of the two-level scan over slab_part
    int2* slab_part;      // [S*R + 1] (starts, candidates) per slab, then their exclusive scan
    int32_t* cand_start;  // [Cmax] sorted global position of the candidate's start hit (S4); the chain is walked in S5
    int32_t* cand_slab;   // [Cmax] instance * R + row of the start hit
    float4* tl_state;     // [6][Cmax] S5: state after the candidate's own hits (fit kernel -> follow kernel)
    float* tl_par;        // [Cmax][5]
    float* tl_cov;        // [Cmax][15]
    float* tl_chi2;       // [Cmax]
    int32_t* tl_nhits;    // [Cmax]  0 = no tracklet
    int32_t* tl_rows;     // [Cmax]  first | last << 8 | ref << 16
    uint16_t* tl_rowhit;  // [Cmax][RP] position in the sorted row of the attached hit (valid in first..last), kNoHit = none
    uint32_t* tl_sel;     // [Cmax][sel_stride] S6 record: kept-row mask, final track index (or ~0), first hit position
    int2* sel_part;       // [Cmax/64 + 2] (tracks, hits) per block of 256 tracklets, then exclusive scan
    int64_t* counts;      // [8] internal copy of the output counts
    int64_t Cmax;
    // phase 2 (k7_phase2.cu), indexed by final track; Tmax = N / sel_min + 1 bounds the tracks (disjoint kept hits)
    int64_t Tmax;
    int32_t* trk_cand;    // [Tmax] candidate id of the final track (written by S6)
    float* p2_par;        // [Tmax][5]  refit of the track's kept hits alone (reading M1)
    float* p2_cov;        // [Tmax][15]
    float* p2_chi2;       // [Tmax]
    int4* p2_info;        // [Tmax] ok, first row, last row, kept hits
    float2* p2_last;      // [Tmax] (y, z) of the outermost kept hit
    int32_t* p2_first;    // [S + 1] first track of every sector instance
    int32_t* p2_rowstart; // [S][R + 1] per sector instance: start in p2_sorted of the fitted tracks that begin in row r
    int32_t* p2_sorted;   // [Tmax] fitted tracks of every sector instance, ordered by their first row
    unsigned long long* p2_best_prev;  // [Tmax] (d2 bits << 32 | predecessor) minimum, ~0 = none
    int32_t* p2_best_next;             // [Tmax]
    int32_t* p2_next;     // [Tmax] links (reading M3)
    int32_t* p2_prev;
    int2* p2_part;        // [Tmax/256 + 2] (heads, chain heads) per block of 256 tracks, then exclusive scan
    int2* p2_chain;       // [Tmax/2 + 1] (innermost segment, merged-track index) of every chain
    int64_t* p2_counts;   // [8] merged tracks, links, failed segment refits, failed chain fits, chains
    // vertex estimate (k8_vertex.cu); n_win = windows of the call, vtx_nb = histogram bins per window
    int32_t* vz_hist;     // [n_win][vtx_nb] z_v histogram of the vertex-like tracks
    int32_t* vz_seed;     // [n_win][64] seed bins, ascending
    int32_t* vz_nseed;    // [n_win + 1] seeds per window, then exclusive scan (vertex index base)
    long long* vz_sum;    // [n_win][64] fixed-point sums of z_v around the seed (deterministic integer atomics)
    int32_t* vz_cnt;      // [n_win][64]
    uint8_t* vz_like;     // [Tmax] 1 = vertex-like, 2 = fitted
    int64_t* vz_counts;   // [2]
    int32_t n_win;
};

struct Problem {
    const void* clusters;  // [n_clusters] records of `layout`
    int layout;            // TPC_INPUT_XYZW (float4), TPC_INPUT_YZ (float2) or TPC_INPUT_I16 (short2)
    const int32_t* row_offsets;
    int32_t n_inst;
    int64_t n_clusters;
};

__host__ __device__ inline int div_up(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// z bin of the per-row grid.  Monotone non-decreasing in z (one rounded subtraction, one rounded multiplication by
// a positive constant, floor, clamp), which is all the superset arguments of S2 and S5 need.
__device__ __forceinline__ int zbin(float z, float z0, float inv_cz, int nz) {
    int b = __float2int_rd(__fmul_rn(__fsub_rn(z, z0), inv_cz));
    return min(max(b, 0), nz - 1);
}

// y strip of the per-row grid: same construction, so monotone non-decreasing in y.
__device__ __forceinline__ int ybin(float y, float y0, float inv_sy, int ny) {
    int b = __float2int_rd(__fmul_rn(__fsub_rn(y, y0), inv_sy));
    return min(max(b, 0), ny - 1);
}

__device__ __forceinline__ float grid_z0(const DevGeom& g, int inst) {
    return (((inst + g.inst_phase) % g.spe) >= g.spe_half) ? g.z0_c : g.z0_a;
}

// ---- launchers (one per stage; each returns the number of kernels it enqueued) ----
int launch_bin_rows(const DevGeom& g, const Workspace& w, const Problem& p, cudaStream_t s);
int launch_neighbours(const DevGeom& g, const Workspace& w, const Problem& p, cudaStream_t s);
struct ChainOut {  // optional user-facing S4 outputs (NULL = skip)
    int32_t* start_hits;
    int64_t start_cap;
    int32_t* cand_hits;
    int32_t* cand_n;
    int64_t cand_cap;
};
int launch_chains(const DevGeom& g, const Workspace& w, const Problem& p, const ChainOut& u, cudaStream_t s);
void launch_scan_int2(int2* part, const int64_t* m_dev, int64_t m_div, int64_t m_cap, int64_t m_host, int64_t* counts,
                      int c0, int c1, cudaStream_t s);
// parity/debug: a link array of the workspace (sorted space) as input-order indices; dir = row offset of the targets
// `mutual`: NULL, or the opposite raw link array -- the link is exported only if it is mutual (cleaned on the fly)
int launch_export_links(const DevGeom& g, const Workspace& w, const Problem& p, const int32_t* link,
                        const int32_t* mutual, int dir, int32_t* out, cudaStream_t s);
int launch_fit(const DevGeom& g, const Workspace& w, const Problem& p, const ChainOut& u, bool count_work, cudaStream_t s);
int launch_follow(const DevGeom& g, const Workspace& w, const Problem& p, int n_sm, bool count_work, cudaStream_t s);

struct SelectOut {  // mirrors the S6 part of tpc_output_t
    float *trk_params, *trk_cov, *trk_chi2, *trk_xref;
    int32_t *trk_cand_id, *trk_nhits, *trk_sector;
    int64_t* trk_hit_offset;
    int32_t* trk_hits;
    int64_t trk_capacity, trk_hits_capacity;
    int32_t* cluster_owner;
    int64_t* counts;  // user counts (device)
};
int launch_select(const DevGeom& g, const Workspace& w, const Problem& p, const SelectOut& o, cudaStream_t s);
// expands the compact tracklet hit table into global indices [Cmax_out][R] (parity/debug output)
struct Phase2Out {  // mirrors tpc_phase2_output_t
    int32_t *seg_next, *seg_prev, *seg_ok;
    float *seg_params, *seg_cov, *seg_chi2;
    int32_t *mtrk_first, *mtrk_nseg, *mtrk_nhits, *mtrk_ok;
    float *mtrk_params, *mtrk_cov, *mtrk_chi2;
    int64_t mtrk_capacity;
    int64_t* counts2;
};
int launch_phase2(const DevGeom& g, const Workspace& w, const Problem& p, const Phase2Out& o, cudaStream_t s);
struct VertexOut {  // mirrors tpc_vertex_output_t
    float *trk_zv, *trk_dca;
    int32_t* trk_vtx;
    float* vtx_z;
    int32_t *vtx_window, *vtx_ntracks;
    int64_t vtx_capacity;
    int64_t* counts3;
};
int launch_vertices(const DevGeom& g, const Workspace& w, const Problem& p, const Phase2Out& m, const VertexOut& o,
                    cudaStream_t s);
int launch_export_tracklets(const DevGeom& g, const Workspace& w, const Problem& p, int32_t* tl_hits, int32_t* tl_rows,
                            int64_t cap, cudaStream_t s);

}  // namespace tpc
