// Incremental network of the streaming state (stream_net.cu): one cluster kernel per update.
#pragma once
#include <vector>
#include "common.cuh"

struct af_stream_net;

// Rows per layer and update of the incremental form: head rows e, tail rows f and new stream rows of every layer of a
// stem-conv / pool / convs / head table at `stride` samples per update (host arithmetic only).  false + *why if the table
// or the stride cannot be run that way.
bool af_stream_net_plan_rows(const std::vector<LayerDesc>& table, int stride, std::vector<int>* e, std::vector<int>* f,
                             std::vector<int>* n_new, const char** why);
// *out = nullptr (and AFRAME_OK) when the configuration does not qualify (*why says which rule); errors are CUDA / memory failures
aframe_status af_stream_net_create(aframe_ctx* ctx, const aframe_weights* w, af_stream_net** out, const char** why);
aframe_status af_stream_net_reset(aframe_ctx* ctx, af_stream_net* sn);
void af_stream_net_free(af_stream_net* sn);
// scores the window d_white [C][K] (fp32, the newest K whitened samples) of this update; no-op while *d_has_filter == 0
aframe_status af_stream_net_launch(aframe_ctx* ctx, af_stream_net* sn, const float* d_white, const int64_t* d_n,
                                   const int* d_has_filter, const int32_t* d_n_scores, float* d_scores);
int af_stream_net_cluster(const af_stream_net* sn);
