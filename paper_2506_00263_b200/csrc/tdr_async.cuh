// tdr_async.cuh — asynchronous remapping: placeholder until the persistent kernel lands.
#pragma once
#include "tdr_stack.cuh"
struct tdr_problem;
struct AsyncMem { u32 *links; u64 *queues; u64 n_links; };
struct Carver;
template <class C> static void async_layout(C &, u64, int, AsyncMem &am) { am.links = nullptr; am.queues = nullptr; am.n_links = 0; }
template <bool CE> static int run_async(tdr_problem *, DevRun &) { return TDR_EINVAL; }
