// tdr_split.cuh — decomposed task scheme under the stack scheme: placeholder until the kernels land.
#pragma once
#include "tdr_stack.cuh"
struct tdr_problem;
struct SplitGrids { int g[EV_COUNT]; };
template <bool CE> static void split_grids(tdr_problem *, size_t, SplitGrids &) {}
template <bool CE> static int split_iteration(tdr_problem *, DevRun &, size_t, const SplitGrids &) { return TDR_EINVAL; }
