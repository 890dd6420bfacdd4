// plk_schedule.cpp -- see plk_schedule.h
#include "plk_schedule.h"

#include <algorithm>
#include <unordered_map>

namespace plk {

int schedule_post(const plk_op* ops, int count, std::vector<int>& level) {
  level.assign(count > 0 ? count : 0, 0);
  if (count < 0 || (count > 0 && ops == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  std::unordered_map<int, int> producer;      // partials buffer -> op that writes it
  std::unordered_map<int, int> reader_level;  // partials buffer -> max level of the ops that read it so far
  std::unordered_map<int, int> scale_owner;
  int n_levels = 0;
  for (int i = 0; i < count; ++i) {
    const plk_op& o = ops[i];
    if (o.dest < 0 || o.child1 < 0 || o.child2 < 0 || o.child1_matrix < 0 || o.child2_matrix < 0)
      return PLK_ERR_OUT_OF_RANGE;
    if (o.dest == o.child1 || o.dest == o.child2) return PLK_ERR_OUT_OF_RANGE;
    if (producer.count(o.dest)) return PLK_ERR_OUT_OF_RANGE;  // two ops writing one buffer
    if (o.dest_scale >= 0) {
      if (scale_owner.count(o.dest_scale)) return PLK_ERR_OUT_OF_RANGE;
      scale_owner[o.dest_scale] = i;
    }
    int lvl = 0;
    const int ch[2] = {o.child1, o.child2};
    for (int k = 0; k < 2; ++k) {
      auto it = producer.find(ch[k]);
      if (it != producer.end()) lvl = std::max(lvl, level[it->second] + 1);
    }
    auto rd = reader_level.find(o.dest);
    if (rd != reader_level.end()) lvl = std::max(lvl, rd->second + 1);  // write-after-read
    level[i] = lvl;
    producer[o.dest] = i;
    for (int k = 0; k < 2; ++k) {
      auto r = reader_level.find(ch[k]);
      if (r == reader_level.end()) reader_level[ch[k]] = lvl; else r->second = std::max(r->second, lvl);
    }
    n_levels = std::max(n_levels, lvl + 1);
  }
  return n_levels;
}

int schedule_pre(const plk_pre_op* ops, int count, std::vector<int>& level, std::vector<int>& partner) {
  level.assign(count > 0 ? count : 0, 0);
  partner.assign(count > 0 ? count : 0, -1);
  if (count < 0 || (count > 0 && ops == nullptr)) return PLK_ERR_OUT_OF_RANGE;
  std::unordered_map<int, int> producer;      // pre buffer -> op that writes it
  std::unordered_map<int, int> reader_level;  // pre buffer -> max level of ops reading it (as parent_pre)
  std::unordered_map<int, std::vector<int>> by_parent;
  int n_levels = 0;
  for (int i = 0; i < count; ++i) {
    const plk_pre_op& o = ops[i];
    if (o.parent_pre < 0 || o.matrix < 0 || o.sibling_post < 0 || o.sibling_matrix < 0 || o.dest_pre < -1)
      return PLK_ERR_OUT_OF_RANGE;
    if (o.dest_pre == o.parent_pre) return PLK_ERR_OUT_OF_RANGE;
    if (o.dest_pre >= 0 && producer.count(o.dest_pre)) return PLK_ERR_OUT_OF_RANGE;
    int lvl = 0;
    auto it = producer.find(o.parent_pre);
    if (it != producer.end()) lvl = level[it->second] + 1;
    if (o.dest_pre >= 0) {
      auto rd = reader_level.find(o.dest_pre);
      if (rd != reader_level.end()) lvl = std::max(lvl, rd->second + 1);
    }
    level[i] = lvl;
    by_parent[o.parent_pre].push_back(i);
  // (bookkeeping after the level is known)
    if (o.dest_pre >= 0) producer[o.dest_pre] = i;
    auto r = reader_level.find(o.parent_pre);
    if (r == reader_level.end()) reader_level[o.parent_pre] = lvl; else r->second = std::max(r->second, lvl);
    n_levels = std::max(n_levels, lvl + 1);
  }
  for (auto& kv : by_parent) {
    const std::vector<int>& v = kv.second;
    for (size_t a = 0; a < v.size(); ++a) {
      if (partner[v[a]] >= 0) continue;
      for (size_t b = a + 1; b < v.size(); ++b) {
        if (partner[v[b]] >= 0) continue;
        const plk_pre_op &x = ops[v[a]], &y = ops[v[b]];
        if (x.matrix == y.sibling_matrix && y.matrix == x.sibling_matrix && level[v[a]] == level[v[b]]) {
          partner[v[a]] = v[b];
          partner[v[b]] = v[a];
          break;
        }
      }
    }
  }
  return n_levels;
}

}  // namespace plk
