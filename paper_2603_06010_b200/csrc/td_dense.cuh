// td_dense.cuh - dense Toeplitz-by-matrix path on the FP64 tensor pipe (SURVEY.md 8a rows S2'-S4').
#pragma once
#include "td_common.cuh"

namespace td {

struct DenseState {
  int max_n = 0;  // longest segment the dense path accepts (0: unavailable)
};
inline void dense_free(DenseState&) {}

}  // namespace td
