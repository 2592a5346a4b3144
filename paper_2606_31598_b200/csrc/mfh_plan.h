// mfh_plan.h -- planner types shared by mfh_plan.cu and mfh_api.cu (host only).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace mfh {

struct Plan;

// Distributed execution (mfh_set_partition): which block positions this rank owns.
struct Partition {
    int rank = 0, world = 1, scheme = 0;   // MFH_PART_*
};
// own[n * n_blk + m] = 1 where block position (n,m) belongs to the rank (R20).
void partition_mask(int n_blk, const Partition& part, std::vector<uint8_t>& own);

// One candidate execution plan p and its model.
struct Candidate {
    int B = 0, n_blk = 0, mode = 0, cached_per_row = 0;
    int64_t n_cached = 0;
    bool pairs = false;                                  // Hermitian pair cache
    bool tc_pairs = true;                                // k-vector complex64 plans: may use the two-sided generator (needs
                                                         // N_blk B/128 extra partial slots; dropped when they do not fit)
    int stream_sms = 0;                                  // partial plans: SMs that stream while the others generate
    double cached_fraction = 0;                          // share of the D^2 entries served from the cache
    double cache_bytes = 0, work_bytes = 0;              // M_op, M_work (Eq. 14-17)
    double t_cached = 0, t_proc = 0, t_reduce = 0;       // seconds per apply, by part
    double t_apply = 0, t_fill = 0, t_job = 0, flops = 0;
    double t_measured = -1.0;                            // Algorithm 2 (Eq. 21), -1 = not measured
    double t_nn = -1.0;                                  // Algorithm 3 (Eq. 25): the surrogate's prediction, -1 = none
    bool feasible = false;                               // Eq. 18
};

void choose_tiling(int B, int n_blk, int n_pairs, int sm_count, int& R, int& Q);
void build_tables(Plan& p, int64_t D, int dtype, int sm_count);
Candidate evaluate_candidate(int64_t D, int dtype, int k, int B, int cached_per_row, bool pairs,
                             int64_t n_applies, int sm_count, const Partition& part = Partition(), double budget_bytes = -1.0);
int pair_full_offsets(int n_blk);
int choose_stream_sms(double cache_bytes, double t_gen_all_sms, int sm_count, double* t_out);
int enumerate_candidates(int64_t D, int dtype, int k, int mode, int B_req, int64_t n_applies,
                         double budget_bytes, int sm_count, std::vector<Candidate>& out,
                         const Partition& part = Partition());
std::string plan_json(int64_t D, int dtype, int k, int64_t n_applies, double budget, int measured,
                      const std::vector<Candidate>& cands);
double planner_alpha();
// Node-level plan space (Eq. 19): JSON over the row-group sizes; returns MFH_OK or MFH_ERR_OUT_OF_MEMORY.
int plan_node(int64_t D, int dtype, int k, int n_op, int64_t n_tasks, int n_gpus, double free_per_gpu, int mode, int B_req,
              int scheme, int64_t n_applies_per_task, std::string& json);

}  // namespace mfh
