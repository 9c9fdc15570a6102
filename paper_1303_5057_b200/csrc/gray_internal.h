// gray_internal.h — shared by the translation units of libgray (not installed, not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/gray.h"

namespace gray {

// Device workspace (gray_workspace_bytes).  One cache line per group to keep the queue head, which
// every warp hits with atomics, away from the counters.
struct Workspace {
  unsigned long long queue_head;          // next photon index to hand out (REFILL schedule)
  unsigned long long pad0[15];
  unsigned long long photon_steps;        // gray_counters
  unsigned long long issued_steps;
  unsigned long long photons_done;
  unsigned long long photons_live;
  unsigned long long fallback_steps;
  unsigned long long pad1[11];
  unsigned long long counts[GRAY_N_STATUS];  // gray_classify: photons per status
  unsigned long long sum_col, sum_row;    // gray_shadow_edge: sums of captured pixel indices
  unsigned int min_col, max_col;          //                   extreme captured columns
  unsigned long long pad2[8];
  double stats[8];                        // gray_shadow_edge: the doubles of gray_shadow_stats
  unsigned long long n_captured;
  unsigned long long pad3[7];
};
static_assert(sizeof(Workspace) == 512, "workspace layout");

void set_error(const char* fmt, ...);
int cuda_fail(cudaError_t e, const char* what);   // records the message, returns GRAY_ERR_CUDA

#define GRAY_CUDA(call)                                       \
  do {                                                        \
    cudaError_t e_ = (call);                                  \
    if (e_ != cudaSuccess) return ::gray::cuda_fail(e_, #call); \
  } while (0)

int check_state(const gray_state* st, bool need_image_fields);
int check_workspace(const void* ws, size_t bytes);
int sm_count();

}  // namespace gray
