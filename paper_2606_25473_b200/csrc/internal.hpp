// Internal declarations shared by the host-side pieces of libattn_jvp (not part of the ABI).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "attn_jvp.h"

namespace aj {

// Thread-local error message behind attn_jvp_last_error().
void set_error(const std::string &msg);
aj_status fail(aj_status st, const std::string &msg);
const char *last_error_cstr();
aj_status check_problem(const aj_problem *p);

struct KeyRange { int32_t k_begin, k_end; int32_t tz = 0; /* tK, tV rows of these keys are structurally zero */ };

// The lowered mask: disjoint query groups, each with sorted, disjoint, merged key ranges.
struct Lowered {
    std::vector<int32_t> q_begin, q_end, range_offset;  // range_offset has num_groups + 1 entries
    std::vector<KeyRange> ranges;
    std::vector<int32_t> q_tz;                          // per group: its tQ rows are structurally zero
    int64_t pairs_per_head = 0;
    int64_t pair_class[3] = {0, 0, 0};                  // pairs needing 2 / 4 / 6 contractions (sum = pairs_per_head)
};

// What the tasks index (aj_task::range_begin / range_count): key ranges with the rows of the query tile that see them.
struct Entries {
    std::vector<int32_t> k_begin, k_end, row_begin, row_end;  // rows relative to the task's q_begin
    std::vector<int32_t> k_tz;                                // tK, tV of the entry's keys are structurally zero
    size_t size() const { return k_begin.size(); }
};

aj_status lower_mask(const aj_problem &p, const aj_mask_desc &m, Lowered &out);
// The lowered mask with the roles of queries and keys swapped (primal backward: dK, dV are accumulated per key tile).
void transpose_lowered(const aj_problem &p, const Lowered &low, Lowered &out);
// Per-group tiling: entries = the lowered ranges, every row of a tile sees every entry of its task.
void build_tasks(const aj_problem &p, const Lowered &low, int32_t tile_q, int32_t tile_k, Entries &ent,
                 std::vector<aj_task> &tasks);
// Packed tiling: query tiles on a global grid; a tile that straddles query groups streams the
// union of their key ranges, each with the interval of its rows that may see it.
void build_tasks_packed(const aj_problem &p, const Lowered &low, int32_t tile_q, int32_t tile_k, Entries &ent,
                        std::vector<aj_task> &tasks);

// Static list scheduling of tasks onto persistent workers (the CTA pairs of the cta_group::2 kernel): off has
// num_workers + 1 entries, worker w runs tasks ids[off[w] .. off[w+1]) in that order.
void assign_workers(const std::vector<aj_task> &tasks, const Entries &ent, int32_t tile_k, int num_workers,
                    std::vector<int32_t> &off, std::vector<int32_t> &ids, bool head_sync = false);

}  // namespace aj

struct aj_schedule {
    aj_problem problem;
    int32_t tile_q, tile_k, tiling;
    aj::Lowered low;
    aj::Entries entries;
    std::vector<aj_task> tasks;
};
