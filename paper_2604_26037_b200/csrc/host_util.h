// host_util.h -- small host helpers shared by the API translation units.
#pragma once
#include "common.h"
#include "cell_tcgen05.h"
#include <new>

template <typename T>
static inline pawfe_status dev_alloc(pawfe_ctx* ctx, T** p, size_t count) {
  *p = nullptr;
  if (count == 0) return PAWFE_OK;
  cudaError_t e = cudaMalloc((void**)p, count * sizeof(T));
  if (e != cudaSuccess) {
    cudaGetLastError();
    ctx->err = std::string("cudaMalloc of ") + std::to_string(count * sizeof(T)) + " bytes: " + cudaGetErrorString(e);
    return PAWFE_ENOMEM;
  }
  return PAWFE_OK;
}
#define TRY(x) do { pawfe_status s_ = (x); if (s_ != PAWFE_OK) return s_; } while (0)

template <typename T>
static inline pawfe_status upload(pawfe_ctx* ctx, T** d, const std::vector<T>& h) {
  TRY(dev_alloc(ctx, d, h.size()));
  CUDA_TRY(ctx, cudaMemcpy(*d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
  return PAWFE_OK;
}

// Raise (never lower) a kernel's dynamic shared-memory limit to `bytes`.  One table for the whole library: a template
// kernel instantiated in several translation units is ONE function to the runtime, so per-unit bookkeeping would let
// one unit lower what another has raised.  func: the kernel's host address.
pawfe_status pawfe_ensure_smem(pawfe_ctx* c, const void* func, size_t bytes);

void pawfe_free_mesh(pawfe_ctx* c);
void pawfe_free_pot(pawfe_ctx* c);
void pawfe_free_atoms(pawfe_ctx* c);

// CUDA-event bracket around one cell-contraction launch (only when pawfe_cell_timing enabled it)
static inline void prof_begin(pawfe_ctx* c) {
  if (!c->prof_on) return;
  if (c->prof_used + 2 > c->prof_ev.size()) {
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    c->prof_ev.push_back(a); c->prof_ev.push_back(b);
  }
  cudaEventRecord(c->prof_ev[c->prof_used], c->stream);
}
static inline void prof_end(pawfe_ctx* c) {
  if (!c->prof_on) return;
  cudaEventRecord(c->prof_ev[c->prof_used + 1], c->stream);
  c->prof_used += 2;
}

// the same around the residual set-up of a filter call (Alg. 2 steps 2-3): bench.py's recurrence-only figure
static inline void prof_setup_mark(pawfe_ctx* c, bool begin) {
  if (!c->prof_on) return;
  if (begin && c->prof_setup_used + 2 > c->prof_setup_ev.size()) {
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    c->prof_setup_ev.push_back(a); c->prof_setup_ev.push_back(b);
  }
  if (begin) cudaEventRecord(c->prof_setup_ev[c->prof_setup_used], c->stream);
  else { cudaEventRecord(c->prof_setup_ev[c->prof_setup_used + 1], c->stream); c->prof_setup_used += 2; }
}
