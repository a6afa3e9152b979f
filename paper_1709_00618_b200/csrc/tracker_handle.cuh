// The opaque handle behind tpc_tracker_t (private to the library's host code).
#pragma once
#include <string>

#include "../../include/tpc_tracker.h"
#include "tpc_common.cuh"

struct tpc_tracker {
    tpc::DevGeom g;
    float* d_row_x = nullptr;  // [7][R]: row_x, row_y0, row_inv_sy, row_wu, row_wd, row_su, row_sd
    void* ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    int n_sm = 148;
    float z_lo = 0.0f, z_hi = 0.0f;  // geometry z range of the z >= 0 side
    float y_half_max = 0.0f;         // half-width of the outermost row's y grid (limit of TPC_INPUT_I16)
    int last_launches = 0;
    // the problem of the last tpc_track_sectors call: tpc_merge_refit (phase 2) reads its workspace
    void* last_ws = nullptr;
    size_t last_ws_bytes = 0;
    cudaStream_t last_stream = nullptr;
    int32_t last_first_inst = 0, last_n_inst = 0;
    const int32_t* last_row_offsets = nullptr;
    int64_t last_n_clusters = 0;
    bool timing = false;
    int input_layout = TPC_INPUT_XYZW;  // tpc_set_input_layout
    bool count_work = false;  // S5 work counters counts[6..9] (tpc_set_work_counters)
    cudaEvent_t ev[TPC_TIMING_RING][TPC_N_STAGES + 1] = {};
    bool ev_valid = false;
    int64_t n_calls = 0;  // timed calls so far (ring position = n_calls % TPC_TIMING_RING)
    std::string err;
};

static inline int fail(tpc_tracker* t, int code, const std::string& msg) {
    if (t) t->err = msg;
    return code;
}

// Error text of entry points that have no tracker handle (tpc_start_hits_static): what tpc_last_error(NULL) returns
// on this thread.
void tpc_set_handleless_error(const std::string& msg);


// bytes per cluster of an input layout, and the alignment mask of its base pointer
static inline int64_t layout_bytes(int layout) { return layout == TPC_INPUT_XYZW ? 16 : layout == TPC_INPUT_YZ ? 8 : 4; }

// The body of tpc_track_sectors on an explicit workspace and stream (the pipeline runs chunks concurrently on
// per-slot workspaces).  `timed` = record the per-stage events of tpc_set_stage_timing.
// `first_inst` = job-wide index of instance 0 (its geometric sector is first_inst % sectors_per_event).
int tpc_track_on(tpc_tracker* t, void* ws, size_t ws_bytes, cudaStream_t s, bool timed, int32_t first_inst,
                 const void* clusters, const int32_t* row_offsets, int32_t n_inst, int64_t n_clusters,
                 const tpc_output_t* out);
