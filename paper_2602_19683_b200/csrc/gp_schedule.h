// gp_schedule.h -- host-side construction of the static work-item order the persistent executor
// (gp_exec.cuh) consumes.  Pure C++ (no CUDA): testable on a machine without a GPU.
//
// The tile-task DAG of PAPER.md Fig. 1 (reading A4) is expanded into block-level work items in
// program order, the dependencies the device enforces with version counters are recovered
// explicitly, and a list-scheduling simulation on `workers` virtual SMs (critical-path-first
// priority, per-item cost model) decides the order in which items are handed out.  The order is
// a topological order of the DAG by construction, which is what makes the in-order ticket
// scheme deadlock-free; the simulated timing only has to be roughly right for waits to be short.
// Trailing updates of four consecutive tile columns are merged into one item per block (a constant of the build);
// the priority of an item is the critical-path length of its tile task, so that the items in flight
// share operand panels in L2.
#pragma once
#include <cstdint>
#include <vector>

namespace gpb {

struct SchedItem {   // must match gpb::Item (gp_exec.cuh)
    uint32_t op, gr, gc, q;
};

enum SchedOp : uint32_t {
    S_UPD_L = 0, S_TRSM_L = 1, S_POTRF = 2, S_ROW_L = 3, S_UPD_V = 4, S_ROW_V = 5, S_UPD_S = 6,
};

struct SchedStats {
    double makespan_us = 0.0;       // simulated
    double work_us = 0.0;           // sum of item costs
    double critical_path_us = 0.0;
    int64_t edges = 0;
};

// M = n / tile, nbt = tile / block, Mm = m / tile.  `blk` (32/64/128) selects the cost model.
void build_cholesky_schedule(int M, int nbt, int workers, std::vector<SchedItem>& out, int blk = 128,
                             SchedStats* stats = nullptr, bool simulate = true);
// with_sigma = false leaves out the W = V^T V items (variance-only prediction).
void build_predict_schedule(int M, int Mm, int nbt, int workers, std::vector<SchedItem>& out, int blk = 128,
                            SchedStats* stats = nullptr, bool simulate = true, bool with_sigma = true);

// Step J of the factorisation without its trailing updates (the FP64 half of gp_cholesky_tiled_mixed): POTRF tile task of
// tile (J, J) + the TRSM tile tasks below it, for blocks that already carry J versions; and its replay check.
void build_panel_schedule(int M, int nbt, int J, int workers, std::vector<SchedItem>& out, int blk = 128, SchedStats* stats = nullptr);
bool validate_panel_schedule(const std::vector<SchedItem>& items, int M, int nbt, int J);

// Checks that `items` is a valid execution order (every wait of every item is satisfied by items
// earlier in the list) and that every block ends at its final version.  Used by the CPU tests.
bool validate_schedule(const std::vector<SchedItem>& items, int M, int Mm, int nbt, bool predict, const char** why,
                       bool with_sigma = true);

// 64-bit FNV-1a hash of an item list: identifies the schedule a measurement (e.g. an ncu DRAM-traffic
// capture under profiles/) was taken with.
uint64_t schedule_fingerprint(const std::vector<SchedItem>& items);

}  // namespace gpb
