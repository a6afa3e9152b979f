// C ABI of libtpctrk.so (include/tpc_tracker.h): handle, workspace carving, stage sequencing.
// Host code only; every step of the hot path runs in the kernels of k1..k6.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/tpc_tracker.h"
#include "tpc_common.cuh"
#include "tracker_handle.cuh"

using namespace tpc;

static thread_local std::string g_create_err;

void tpc_set_handleless_error(const std::string& msg) { g_create_err = msg; }

template <typename T>
static T dflt(T v, T d) { return v == (T)0 ? d : v; }

extern "C" int tpc_tracker_create(const tpc_geometry_t* geom, float bz, tpc_tracker_t** out) {
    if (!geom || !out || !geom->row_x) { g_create_err = "NULL argument"; return TPC_ERR_ARG; }
    *out = nullptr;
    const int R = geom->n_rows;
    if (R < 3 || R > kMaxRows) { g_create_err = "n_rows out of [3,255]"; return TPC_ERR_GEOMETRY; }
    // Rows must be strictly increasing.  Equal spacing is no longer required (reading A5'): S2 weights its
    // two first differences by the row steps and scales its window with them; a step within 1e-4 p + 4e-5 cm of the
    // mean pitch p counts as p, so that equally spaced rows keep the arithmetic of the default reading bit for bit.
    const double pitch = ((double)geom->row_x[R - 1] - (double)geom->row_x[0]) / (R - 1);
    if (!(pitch > 0.0)) { g_create_err = "rows not increasing"; return TPC_ERR_GEOMETRY; }
    bool uniform = true;
    for (int r = 1; r < R; r++) {
        const double d = (double)geom->row_x[r] - (double)geom->row_x[r - 1];
        if (!(d > 0.0)) {
            g_create_err = "pad rows must be strictly increasing";
            return TPC_ERR_GEOMETRY;
        }
        if (std::fabs(d - pitch) > 1e-4 * pitch + 4e-5) uniform = false;
    }
    if (!uniform && geom->params.nf_bridge_rows != 0) {
        g_create_err = "nf_bridge_rows (reading A2') is defined for equally spaced pad rows only";
        return TPC_ERR_GEOMETRY;
    }
    if (geom->sectors_per_event < 2 || (geom->sectors_per_event & 1) || !(geom->z_hi > geom->z_lo) ||
        !(geom->sigma_y > 0.0f) || !(geom->sigma_z > 0.0f) || !(geom->half_angle_rad > 0.0f)) {
        g_create_err = "bad sectors_per_event / z range / sigma / half angle";
        return TPC_ERR_ARG;
    }
    const tpc_params_t& p = geom->params;
    tpc_tracker* t = new (std::nothrow) tpc_tracker();
    if (!t) { g_create_err = "out of host memory"; return TPC_ERR_ARG; }
    DevGeom& g = t->g;
    g.R = R;
    g.RP = (R + 7) & ~7;
    g.sel_words = (R + 31) / 32;
    g.sel_stride = (g.sel_words + 2 + 3) & ~3;
    // per-row 2-D grid: ny strips across the row, z bins of cz (performance only, no result depends on either).
    // Default cz = 6.75 cm > 2 * (kf_win_max + the follower's speculation margin), so a search window touches at most
    // 2 z bins.
    int ny = dflt(p.grid_cells_y, 12);
    if (ny < 1) ny = 1;
    if (ny > 64) ny = 64;
    float cz = dflt(p.grid_cell_z, 6.75f);
    int nz = (int)std::ceil(((double)geom->z_hi - (double)geom->z_lo) / cz);
    if (nz < 1) nz = 1;
    if ((int64_t)nz * ny > kMaxCells) {  // too fine: widen the z bins until the row grid fits
        nz = kMaxCells / ny;
        cz = (float)(((double)geom->z_hi - (double)geom->z_lo) / nz);
    }
    g.nz = nz;
    g.ny = ny;
    g.ncell = nz * ny;
    g.nzp = (g.ncell + 1 + 15) & ~15;  // rows of the table start on 32-byte sectors
    g.spe = geom->sectors_per_event;
    g.spe_half = g.spe / 2;
    g.inst_phase = 0;
    g.z0_a = geom->z_lo;
    t->z_lo = geom->z_lo;
    t->z_hi = geom->z_hi;
    g.z0_c = -geom->z_hi;
    g.inv_cz = 1.0f / cz;
    g.nf_wy = dflt(p.nf_win_y, 2.0f);
    g.nf_wz = dflt(p.nf_win_z, 2.5f);
    g.nf_d2max = dflt(p.nf_d2_max, 1.0f);
    g.bridge = p.nf_bridge_rows != 0 ? 1 : 0;
    g.cand_min = dflt(p.cand_min_hits, 4);
    g.cand_max = dflt(p.cand_max_hits, 10);
    const float p0d[5] = {1.0f, 1.0f, 0.1f, 0.1f, 10.0f};
    for (int i = 0; i < 5; i++) g.p0[i] = dflt(p.kf_p0[i], p0d[i]);
    g.gate = dflt(p.kf_gate_sigma, 4.0f);
    g.wmax = dflt(p.kf_win_max, 3.0f);
    g.max_gap = dflt(p.kf_max_gap, 5);
    g.max_s = dflt(p.kf_max_sinphi, 0.95f);
    g.edge_margin = dflt(p.kf_edge_margin, 2.0f);
    g.tan_half = (float)std::tan((double)geom->half_angle_rad);
    g.sel_min = dflt(p.sel_min_hits, 10);
    g.cos_2h = (float)std::cos(2.0 * (double)geom->half_angle_rad);
    g.sin_2h = (float)std::sin(2.0 * (double)geom->half_angle_rad);
    {  // z_v histogram of the vertex estimate: 0.5 cm bins over [-h, h), h = the geometry's |z| range + 50 cm
        const double lo = std::fabs((double)geom->z_lo - 50.0), hi = std::fabs((double)geom->z_hi + 50.0);
        const double h = lo > hi ? lo : hi;
        g.vtx_h = (float)h;
        g.vtx_nb = (int)std::ceil(2.0 * h / 0.5);
    }
    g.sy2 = (float)((double)geom->sigma_y * (double)geom->sigma_y);
    g.sz2 = (float)((double)geom->sigma_z * (double)geom->sigma_z);
    g.cB = (float)(-0.00299792458 * (double)bz);
    if (g.cand_min < 2 || g.cand_max > kCandMax || g.cand_max < g.cand_min || g.cand_max < 3) {
        delete t;
        g_create_err = "cand_min_hits/cand_max_hits out of range (2 <= min <= max <= 10, max >= 3)";
        return TPC_ERR_ARG;
    }
    constexpr int kRowTables = 7;  // row_x, row_y0, row_inv_sy, row_wu, row_wd, row_su, row_sd
    std::vector<float> rows(kRowTables * (size_t)R, 1.0f);
    for (int r = 0; r < R; r++) {
        const float hw = geom->row_x[r] * g.tan_half + 0.5f;  // half-width of the row's y grid
        rows[r] = geom->row_x[r];
        if (hw > t->y_half_max) t->y_half_max = hw;
        rows[R + r] = -hw;
        rows[2 * R + r] = (float)ny / (2.0f * hw);
        if (r >= 1 && r <= R - 2) {  // step factors of reading A5' (rows 0 and R-1 own no links)
            const double up = (double)geom->row_x[r + 1] - (double)geom->row_x[r];
            const double dn = (double)geom->row_x[r] - (double)geom->row_x[r - 1];
            const double tol = 1e-4 * pitch + 4e-5;
            const bool up_reg = std::fabs(up - pitch) <= tol, dn_reg = std::fabs(dn - pitch) <= tol;
            if (!(up_reg && dn_reg)) {
                rows[3 * R + r] = (float)(2.0 * dn / (up + dn));
                rows[4 * R + r] = (float)(2.0 * up / (up + dn));
            }
            if (!up_reg) rows[5 * R + r] = (float)(up / pitch);
            if (!dn_reg) rows[6 * R + r] = (float)(dn / pitch);
        }
    }
    cudaError_t e = cudaMalloc(&t->d_row_x, sizeof(float) * kRowTables * R);
    if (e == cudaSuccess)
        e = cudaMemcpy(t->d_row_x, rows.data(), sizeof(float) * kRowTables * R, cudaMemcpyHostToDevice);
    int dev = 0;
    if (e == cudaSuccess) e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&t->n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) {
        g_create_err = std::string("CUDA: ") + cudaGetErrorString(e);
        if (t->d_row_x) cudaFree(t->d_row_x);
        delete t;
        return TPC_ERR_CUDA;
    }
    g.row_x = t->d_row_x;
    g.row_y0 = t->d_row_x + R;
    g.row_inv_sy = t->d_row_x + 2 * R;
    g.uniform_pitch = uniform ? 1 : 0;
    g.row_wu = t->d_row_x + 3 * R;
    g.row_wd = t->d_row_x + 4 * R;
    g.row_su = t->d_row_x + 5 * R;
    g.row_sd = t->d_row_x + 6 * R;
    *out = t;
    return TPC_OK;
}

extern "C" void tpc_tracker_destroy(tpc_tracker_t* t) {
    if (!t) return;
    if (t->ev_valid)
        for (auto& ring : t->ev)
            for (auto& e : ring) cudaEventDestroy(e);
    if (t->d_row_x) cudaFree(t->d_row_x);
    delete t;
}

// ---- workspace carving: one function computes the layout for both sizing and use ----
namespace {
struct Carver {
    char* base;
    size_t off = 0;
    template <typename T>
    T* take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

size_t carve(const DevGeom& g, void* base, int64_t N, int64_t S, Workspace* w) {
    Carver c{static_cast<char*>(base)};
    const size_t n = (size_t)(N > 0 ? N : 1), slabs = (size_t)(S > 0 ? S : 1) * g.R;
    const size_t cmax = (size_t)(N / g.cand_min + 1);
    Workspace v;
    v.counts = c.take<int64_t>(TPC_N_COUNTS);
    v.hit_yz = c.take<float2>(n);
    v.hit_idx = c.take<uint16_t>(n);
    v.hit_pos = c.take<uint16_t>(n);
    v.bin_start = c.take<uint16_t>(slabs * g.nzp);
    v.up_raw = c.take<int32_t>(n);
    v.dn_raw = c.take<int32_t>(n);
    v.up = c.take<int32_t>(n);
    v.claim = c.take<uint32_t>(n);
    v.flags = c.take<uint8_t>(n);
    v.slab_part = c.take<int2>(slabs + 1);
    v.scan_tmp = c.take<int2>(slabs / 4096 + 2);
    v.cand_start = c.take<int32_t>(cmax);
    v.cand_slab = c.take<int32_t>(cmax);
    v.tl_state = c.take<float4>(cmax * 6);
    v.tl_par = c.take<float>(cmax * 5);
    v.tl_cov = c.take<float>(cmax * 15);
    v.tl_chi2 = c.take<float>(cmax);
    v.tl_nhits = c.take<int32_t>(cmax);
    v.tl_rows = c.take<int32_t>(cmax);
    v.tl_rowhit = c.take<uint16_t>(cmax * g.RP);
    v.tl_sel = c.take<uint32_t>(cmax * g.sel_stride);
    v.sel_part = c.take<int2>(cmax / 64 + 2);
    v.Cmax = (int64_t)cmax;
    const size_t tmax = (size_t)(N / (g.sel_min > 0 ? g.sel_min : 1) + 1);
    v.Tmax = (int64_t)tmax;
    v.trk_cand = c.take<int32_t>(tmax);
    v.p2_par = c.take<float>(tmax * 5);
    v.p2_cov = c.take<float>(tmax * 15);
    v.p2_chi2 = c.take<float>(tmax);
    v.p2_info = c.take<int4>(tmax);
    v.p2_last = c.take<float2>(tmax);
    v.p2_first = c.take<int32_t>((size_t)(S > 0 ? S : 1) + 1);
    v.p2_rowstart = c.take<int32_t>((size_t)(S > 0 ? S : 1) * ((size_t)g.R + 1));
    v.p2_sorted = c.take<int32_t>(tmax);
    v.p2_best_prev = c.take<unsigned long long>(tmax);
    v.p2_best_next = c.take<int32_t>(tmax);
    v.p2_next = c.take<int32_t>(tmax);
    v.p2_prev = c.take<int32_t>(tmax);
    v.p2_part = c.take<int2>(tmax / 256 + 2);
    v.p2_chain = c.take<int2>(tmax / 2 + 1);
    v.p2_counts = c.take<int64_t>(8);
    const size_t nwin = (size_t)(S > 0 ? S : 1) / (size_t)g.spe + 2;
    v.n_win = (int32_t)nwin;
    v.vz_hist = c.take<int32_t>(nwin * (size_t)g.vtx_nb);
    v.vz_seed = c.take<int32_t>(nwin * TPC_VTX_MAX_PER_WINDOW);
    v.vz_nseed = c.take<int32_t>(nwin + 1);
    v.vz_sum = c.take<long long>(nwin * TPC_VTX_MAX_PER_WINDOW);
    v.vz_cnt = c.take<int32_t>(nwin * TPC_VTX_MAX_PER_WINDOW);
    v.vz_like = c.take<uint8_t>(tmax);
    v.vz_counts = c.take<int64_t>(2);
    if (w) *w = v;
    return (c.off + 255) & ~(size_t)255;
}
}  // namespace

extern "C" size_t tpc_workspace_bytes(const tpc_tracker_t* t, int64_t max_clusters, int64_t max_inst) {
    if (!t || max_clusters < 0 || max_inst < 0) return 0;
    return carve(t->g, nullptr, max_clusters, max_inst, nullptr);
}

extern "C" int tpc_set_workspace(tpc_tracker_t* t, void* dev_ptr, size_t bytes) {
    if (!t) return TPC_ERR_ARG;
    if (!dev_ptr || ((uintptr_t)dev_ptr & 255)) return fail(t, TPC_ERR_ARG, "workspace must be non-NULL and 256-byte aligned");
    if (dev_ptr != t->ws || bytes != t->ws_bytes) t->last_ws = nullptr;  // the old workspace may be gone: phase 2 needs a new track call
    t->ws = dev_ptr;
    t->ws_bytes = bytes;
    return TPC_OK;
}

extern "C" int tpc_set_stream(tpc_tracker_t* t, void* s) {
    if (!t) return TPC_ERR_ARG;
    t->stream = static_cast<cudaStream_t>(s);
    return TPC_OK;
}

extern "C" int tpc_set_input_layout(tpc_tracker_t* t, int32_t layout) {
    if (!t) return TPC_ERR_ARG;
    if (layout != TPC_INPUT_XYZW && layout != TPC_INPUT_YZ && layout != TPC_INPUT_I16)
        return fail(t, TPC_ERR_ARG, "unknown input layout");
    if (layout == TPC_INPUT_I16 && ((double)t->z_hi - (double)t->z_lo) > 65535.0 * (double)TPC_I16_Z_STEP)
        return fail(t, TPC_ERR_ARG, "TPC_INPUT_I16 covers 1024 cm of z; the geometry's z range is wider");
    if (layout == TPC_INPUT_I16 && !(t->y_half_max < 32768.0f * TPC_I16_Y_STEP))
        return fail(t, TPC_ERR_ARG, "TPC_INPUT_I16 covers |y| < 128 cm; the outermost pad row is wider");
    t->input_layout = layout;
    return TPC_OK;
}

extern "C" int tpc_set_work_counters(tpc_tracker_t* t, int32_t enable) {
    if (!t) return TPC_ERR_ARG;
    t->count_work = enable != 0;
    return TPC_OK;
}

extern "C" int tpc_set_stage_timing(tpc_tracker_t* t, int32_t enable) {
    if (!t) return TPC_ERR_ARG;
    if (enable && !t->ev_valid) {
        for (auto& ring : t->ev)
            for (auto& e : ring)
                if (cudaEventCreate(&e) != cudaSuccess) return fail(t, TPC_ERR_CUDA, "cudaEventCreate failed");
        t->ev_valid = true;
    }
    t->timing = enable != 0;
    return TPC_OK;
}

extern "C" int tpc_stage_times_ms(tpc_tracker_t* t, int32_t age, float* out_ms) {
    if (!t || !out_ms) return TPC_ERR_ARG;
    if (!t->ev_valid) return fail(t, TPC_ERR_ARG, "stage timing was not enabled");
    if (age < 0 || age >= TPC_TIMING_RING || age >= t->n_calls) return fail(t, TPC_ERR_ARG, "no timed call of that age");
    cudaEvent_t* ev = t->ev[(t->n_calls - 1 - age) % TPC_TIMING_RING];
    cudaError_t e = cudaEventSynchronize(ev[TPC_N_STAGES]);
    for (int i = 0; i < TPC_N_STAGES && e == cudaSuccess; i++) e = cudaEventElapsedTime(&out_ms[i], ev[i], ev[i + 1]);
    if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
    return TPC_OK;
}

extern "C" int tpc_track_sectors(tpc_tracker_t* t, const void* clusters, const int32_t* row_offsets, int32_t n_inst,
                                 int64_t n_clusters, const tpc_output_t* out) {
    if (!t) return TPC_ERR_ARG;
    return tpc_track_on(t, t->ws, t->ws_bytes, t->stream, true, 0, clusters, row_offsets, n_inst, n_clusters, out);
}

int tpc_track_on(tpc_tracker* t, void* ws, size_t ws_bytes, cudaStream_t s, bool timed, int32_t first_inst,
                 const void* clusters, const int32_t* row_offsets, int32_t n_inst, int64_t n_clusters,
                 const tpc_output_t* out) {
    if (!out || !out->counts) return fail(t, TPC_ERR_ARG, "out and out->counts are required");
    if (n_inst < 0 || n_clusters < 0 || n_clusters >= ((int64_t)1 << 31)) return fail(t, TPC_ERR_ARG, "bad sizes");
    if ((int64_t)n_inst * t->g.R + 1 >= ((int64_t)1 << 31)) return fail(t, TPC_ERR_ARG, "too many sector instances");
    // the follower addresses the cell table by its 32-byte row units in 32 bits (a table beyond 2^32 units = 137 GB
    // does not fit the workspace anyway)
    if ((int64_t)n_inst * t->g.R * (t->g.nzp >> 4) >= ((int64_t)1 << 32))
        return fail(t, TPC_ERR_ARG, "too many sector instances for this grid");
    if (n_clusters > 0 && (!clusters || n_inst == 0)) return fail(t, TPC_ERR_ARG, "NULL input");
    if (n_inst > 0 && !row_offsets) return fail(t, TPC_ERR_ARG, "row_offsets is required when n_sector_instances > 0");
    if ((uintptr_t)clusters & (uintptr_t)(layout_bytes(t->input_layout) - 1))
        return fail(t, TPC_ERR_ARG, "clusters must be aligned to one record (16 / 8 / 4 bytes for XYZW / YZ / I16)");
    Workspace w;
    const size_t need = carve(t->g, ws, n_clusters, n_inst, &w);
    if (!ws || need > ws_bytes) return fail(t, TPC_ERR_WORKSPACE, "workspace missing or too small");
    DevGeom g = t->g;
    g.inst_phase = first_inst % g.spe;
    Problem p{clusters, t->input_layout, row_offsets, n_inst, n_clusters};
    int launches = 0;
    const bool tm = timed && t->timing && t->ev_valid;
    cudaEvent_t* ev = t->ev[t->n_calls % TPC_TIMING_RING];
    if (tm) t->n_calls++;
    cudaMemsetAsync(w.counts, 0, sizeof(int64_t) * TPC_N_COUNTS, s);
    if (out->cluster_owner && n_clusters > 0) cudaMemsetAsync(out->cluster_owner, 0xFF, sizeof(int32_t) * n_clusters, s);
    if (tm) cudaEventRecord(ev[0], s);
    launches += launch_bin_rows(g, w, p, s);
    if (tm) cudaEventRecord(ev[1], s);
    launches += launch_neighbours(g, w, p, s);
    if (tm) cudaEventRecord(ev[2], s);
    ChainOut co{out->start_hits, out->start_hits ? out->start_capacity : 0, out->cand_hits, out->cand_n,
                (out->cand_hits || out->cand_n) ? out->cand_capacity : 0};
    launches += launch_chains(g, w, p, co, s);
    if (tm) cudaEventRecord(ev[3], s);
    launches += launch_fit(g, w, p, co, t->count_work, s);
    if (tm) cudaEventRecord(ev[4], s);
    launches += launch_follow(g, w, p, t->n_sm, t->count_work, s);
    if (tm) cudaEventRecord(ev[5], s);
    SelectOut so{out->trk_params, out->trk_cov, out->trk_chi2, out->trk_xref, out->trk_cand_id, out->trk_nhits,
                 out->trk_sector, out->trk_hit_offset, out->trk_hits, out->trk_capacity, out->trk_hits_capacity,
                 out->cluster_owner, out->counts};
    launches += launch_select(g, w, p, so, s);
    if (tm) cudaEventRecord(ev[6], s);
    // optional parity/debug copies (device to device, same stream)
    if (n_clusters > 0) {
        launches += launch_export_links(g, w, p, w.up_raw, nullptr, +1, out->link_up_raw, s);
        launches += launch_export_links(g, w, p, w.dn_raw, nullptr, -1, out->link_dn_raw, s);
        launches += launch_export_links(g, w, p, w.up, nullptr, +1, out->link_up, s);
        launches += launch_export_links(g, w, p, w.dn_raw, w.up_raw, -1, out->link_dn, s);  // cleaned on the fly
        const int64_t tc = out->tl_capacity < w.Cmax ? out->tl_capacity : w.Cmax;
        if (tc > 0) {
            if (out->tl_params) cudaMemcpyAsync(out->tl_params, w.tl_par, sizeof(float) * 5 * tc, cudaMemcpyDeviceToDevice, s);
            if (out->tl_cov) cudaMemcpyAsync(out->tl_cov, w.tl_cov, sizeof(float) * 15 * tc, cudaMemcpyDeviceToDevice, s);
            if (out->tl_chi2) cudaMemcpyAsync(out->tl_chi2, w.tl_chi2, sizeof(float) * tc, cudaMemcpyDeviceToDevice, s);
            if (out->tl_nhits) cudaMemcpyAsync(out->tl_nhits, w.tl_nhits, sizeof(int32_t) * tc, cudaMemcpyDeviceToDevice, s);
            launches += launch_export_tracklets(g, w, p, out->tl_hits, out->tl_rows, tc, s);
        }
    }
    t->last_launches = launches;
    if (timed) {  // a user call: phase 2 may follow.  The pipeline's chunks (timed == false) leave no such state.
        t->last_ws = ws;
        t->last_ws_bytes = ws_bytes;
        t->last_stream = s;
        t->last_first_inst = first_inst;
        t->last_row_offsets = row_offsets;
        t->last_n_inst = n_inst;
        t->last_n_clusters = n_clusters;
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
    return TPC_OK;
}

extern "C" int tpc_merge_refit(tpc_tracker_t* t, const tpc_phase2_output_t* out) {
    if (!t) return TPC_ERR_ARG;
    if (!out || !out->counts2) return fail(t, TPC_ERR_ARG, "out and out->counts2 are required");
    if (!t->last_ws) return fail(t, TPC_ERR_ARG, "tpc_merge_refit needs a preceding tpc_track_sectors call on this tracker");
    Workspace w;
    carve(t->g, t->last_ws, t->last_n_clusters, t->last_n_inst, &w);
    DevGeom g = t->g;
    g.inst_phase = t->last_first_inst % g.spe;
    Problem p{nullptr, t->input_layout, t->last_row_offsets, t->last_n_inst, t->last_n_clusters};
    const Phase2Out o{out->seg_next, out->seg_prev, out->seg_ok, out->seg_params, out->seg_cov, out->seg_chi2,
                      out->mtrk_first, out->mtrk_nseg, out->mtrk_nhits, out->mtrk_ok, out->mtrk_params, out->mtrk_cov,
                      out->mtrk_chi2, out->mtrk_capacity, out->counts2};
    t->last_launches = launch_phase2(g, w, p, o, t->last_stream);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
    return TPC_OK;
}

extern "C" int tpc_estimate_vertices(tpc_tracker_t* t, const tpc_phase2_output_t* m, const tpc_vertex_output_t* out) {
    if (!t) return TPC_ERR_ARG;
    if (!out || !out->counts3 || !out->trk_zv) return fail(t, TPC_ERR_ARG, "out, out->counts3 and out->trk_zv are required");
    if (!m || !m->mtrk_first || !m->mtrk_nhits || !m->mtrk_ok || !m->mtrk_params || !m->counts2)
        return fail(t, TPC_ERR_ARG, "merged: mtrk_first, mtrk_nhits, mtrk_ok, mtrk_params and counts2 are required");
    if (!t->last_ws) return fail(t, TPC_ERR_ARG, "tpc_estimate_vertices needs preceding tpc_track_sectors + tpc_merge_refit calls");
    if ((size_t)t->g.vtx_nb * sizeof(int32_t) > kVtxMaxSmemBytes)
        return fail(t, TPC_ERR_ARG, "the geometry's z range is too wide for the vertex histogram (0.5 cm bins in shared memory)");
    Workspace w;
    carve(t->g, t->last_ws, t->last_n_clusters, t->last_n_inst, &w);
    DevGeom g = t->g;
    g.inst_phase = t->last_first_inst % g.spe;
    Problem p{nullptr, t->input_layout, t->last_row_offsets, t->last_n_inst, t->last_n_clusters};
    const Phase2Out mo{m->seg_next, m->seg_prev, m->seg_ok, m->seg_params, m->seg_cov, m->seg_chi2, m->mtrk_first,
                       m->mtrk_nseg, m->mtrk_nhits, m->mtrk_ok, m->mtrk_params, m->mtrk_cov, m->mtrk_chi2,
                       m->mtrk_capacity, m->counts2};
    const VertexOut vo{out->trk_zv, out->trk_dca, out->trk_vtx, out->vtx_z, out->vtx_window, out->vtx_ntracks,
                       out->vtx_capacity, out->counts3};
    t->last_launches = launch_vertices(g, w, p, mo, vo, t->last_stream);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(t, TPC_ERR_CUDA, std::string("CUDA: ") + cudaGetErrorString(e));
    return TPC_OK;
}

extern "C" int tpc_check_counts(const int64_t* c, const tpc_output_t* out) {
    if (!c || !out) return TPC_ERR_ARG;
    if (c[5] != 0) return TPC_ERR_INPUT;
    if (out->start_hits && c[0] > out->start_capacity) return TPC_ERR_CAPACITY;
    if ((out->cand_hits || out->cand_n) && c[1] > out->cand_capacity) return TPC_ERR_CAPACITY;
    if ((out->tl_params || out->tl_cov || out->tl_chi2 || out->tl_nhits || out->tl_rows || out->tl_hits) &&
        c[1] > out->tl_capacity)
        return TPC_ERR_CAPACITY;
    if (c[3] > out->trk_capacity && (out->trk_params || out->trk_cov || out->trk_chi2 || out->trk_xref ||
                                     out->trk_cand_id || out->trk_nhits || out->trk_sector || out->trk_hit_offset ||
                                     out->trk_hits || out->cluster_owner))
        return TPC_ERR_CAPACITY;
    if (out->trk_hits && c[4] > out->trk_hits_capacity) return TPC_ERR_CAPACITY;
    return TPC_OK;
}

extern "C" int32_t tpc_last_launch_count(const tpc_tracker_t* t) { return t ? t->last_launches : 0; }

extern "C" const char* tpc_last_error(const tpc_tracker_t* t) { return t ? t->err.c_str() : g_create_err.c_str(); }
