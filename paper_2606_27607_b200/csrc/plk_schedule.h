// plk_schedule.h -- host-side grouping of operation lists into dependency levels ("level-batched from
// an operation list"; section 7 step 2).  Pure C++, no CUDA; also exported through plk_schedule_levels /
// plk_schedule_pre_levels so that the logic is testable without a GPU.
#pragma once
#include <vector>

#include "../../include/plk.h"

namespace plk {

// level[i] = 0 when ops[i] depends on no earlier op of the list, else 1 + max level of the ops it depends on.
// Dependencies: a child produced by an earlier op (read-after-write) and a dest read by an earlier op
// (write-after-read).  Returns the number of levels, or a negative plk_status.
int schedule_post(const plk_op* ops, int count, std::vector<int>& level);

// Pre-order: dependency = parent_pre (or, WAR, dest_pre) touched by an earlier op.  partner[i] = the other op with
// the same parent_pre whose (matrix, sibling_matrix) are the mirror image of ops[i]'s -- the two children of one
// parent, fused into one launch item -- or -1.  Partners always share a level.
int schedule_pre(const plk_pre_op* ops, int count, std::vector<int>& level, std::vector<int>& partner);

}  // namespace plk
