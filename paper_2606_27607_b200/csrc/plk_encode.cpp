// plk_encode.cpp -- tip-state encoding and unique-site-pattern compression (SURVEY 8(a) step 0
// "unique site patterns").  Integer work on the host, done once per alignment before anything is uploaded; rules:
// SURVEY 8(c) rows 7, 16, 17 (restated in include/plk.h).
#include <cstring>
#include <vector>

#include "../../include/plk.h"

namespace {

inline int base_code(char ch) {
  switch (ch) {
    case 'A': case 'a': return 0;
    case 'C': case 'c': return 1;
    case 'G': case 'g': return 2;
    case 'T': case 't': case 'U': case 'u': return 3;
    default: return -1;
  }
}

// sense-codon index of idx64 = 16 n1 + 4 n2 + n3 (A<C<G<T); the stops TAA (48), TAG (50), TGA (56) give -1
inline int sense_index(int idx64) {
  if (idx64 == 48 || idx64 == 50 || idx64 == 56) return -1;
  return idx64 - (idx64 > 48) - (idx64 > 50) - (idx64 > 56);
}

inline uint64_t hash_column(const uint8_t* col, int n) {
  uint64_t h = 1469598103934665603ull;  // FNV-1a
  for (int i = 0; i < n; ++i) {
    h ^= col[i];
    h *= 1099511628211ull;
  }
  return h;
}

}  // namespace

extern "C" int plk_encode_and_compress(int state_kind, int taxa, int64_t sites, const char* const* seqs,
                                       uint8_t* out_states, double* out_weights, int64_t* out_site_to_pattern,
                                       int64_t* out_pattern_count) {
  if (taxa <= 0 || sites < 0 || seqs == nullptr || out_states == nullptr || out_weights == nullptr ||
      out_site_to_pattern == nullptr || out_pattern_count == nullptr)
    return PLK_ERR_OUT_OF_RANGE;
  if (state_kind != PLK_NUCLEOTIDE && state_kind != PLK_CODON) return PLK_ERR_UNSUPPORTED;
  if (state_kind == PLK_CODON && sites % 3 != 0) return PLK_ERR_OUT_OF_RANGE;
  const int64_t cols = state_kind == PLK_CODON ? sites / 3 : sites;
  *out_pattern_count = 0;
  if (cols == 0) return PLK_SUCCESS;

  // 1. encode, column-major: code[col][taxon]
  std::vector<uint8_t> code((size_t)cols * taxa);
  for (int t = 0; t < taxa; ++t) {
    const char* s = seqs[t];
    if (s == nullptr) return PLK_ERR_OUT_OF_RANGE;
    for (int64_t j = 0; j < cols; ++j) {
      uint8_t v;
      if (state_kind == PLK_NUCLEOTIDE) {
        const int b = base_code(s[j]);
        v = (uint8_t)(b < 0 ? 4 : b);
      } else {
        const int b1 = base_code(s[3 * j]), b2 = base_code(s[3 * j + 1]), b3 = base_code(s[3 * j + 2]);
        if (b1 < 0 || b2 < 0 || b3 < 0) {
          v = 61;
        } else {
          const int idx = sense_index(16 * b1 + 4 * b2 + b3);
          if (idx < 0) return PLK_ERR_STOP_CODON;
          v = (uint8_t)idx;
        }
      }
      code[(size_t)j * taxa + t] = v;
    }
  }

  // 2. merge identical columns, numbering patterns by first occurrence (open-addressing table of pattern ids)
  size_t cap = 16;
  while (cap < (size_t)cols * 2) cap <<= 1;
  std::vector<int64_t> table(cap, -1);
  std::vector<int64_t> first_col;  // pattern -> first column showing it
  int64_t n_pat = 0;
  for (int64_t j = 0; j < cols; ++j) {
    const uint8_t* col = &code[(size_t)j * taxa];
    size_t h = (size_t)hash_column(col, taxa) & (cap - 1);
    int64_t id = -1;
    while (table[h] >= 0) {
      const int64_t cand = table[h];
      if (std::memcmp(&code[(size_t)first_col[cand] * taxa], col, (size_t)taxa) == 0) {
        id = cand;
        break;
      }
      h = (h + 1) & (cap - 1);
    }
    if (id < 0) {
      id = n_pat++;
      table[h] = id;
      first_col.push_back(j);
      out_weights[id] = 0.0;
      for (int t = 0; t < taxa; ++t) out_states[(size_t)t * cols + id] = col[t];
    }
    out_weights[id] += 1.0;
    out_site_to_pattern[j] = id;
  }
  *out_pattern_count = n_pat;
  return PLK_SUCCESS;
}
