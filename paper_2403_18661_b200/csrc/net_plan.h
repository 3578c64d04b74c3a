// Activation-slot plan: each layer output lives in one of a few equally sized slots, reused after its
// last consumer (a ResNet needs three to four).
#pragma once
#include <stddef.h>
#include <stdint.h>
#include "../../include/aframe.h"
#include <vector>

struct aframe_weights;
struct aframe_ctx;

struct NetPlan {
  std::vector<int> slot;       // per layer: slot index, -1 if the output is never materialised
  std::vector<size_t> elems;   // per layer: output elements per window
  int n_slots = 0;
  size_t slot_elems = 0;       // elements per window of the largest output
};

bool af_make_plan(const aframe_weights* w, bool fuse_stem_pool, NetPlan& plan);
aframe_status af_launch_head(aframe_ctx* ctx, const void* d_in, int in_dt, const float* d_w, float bias, int T, int C,
                             int64_t B, float* d_scores);
