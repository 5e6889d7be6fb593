// grpic_step_host: one full PIC step with the particle state in HOST memory (the end-to-end
// entry of the library).  The particle SoA is streamed through the GPU in chunks on three
// streams -- host->device copy of chunk c+1, fused push+deposit+compaction of chunk c and
// device->host copy of chunk c-1 overlap, so the step costs about max(H2D, D2H) of the particle
// state instead of their sum -- then the flux is finalised, the field step runs on the device
// and J is copied back.  Every arithmetic step is the same kernels the device-resident calls use.
#include <new>

#include "grpic_internal.cuh"

namespace {

constexpr int kBufs = 2;

struct HostStepState {
  int64_t chunk = 0;                 // particles per chunk the buffers were sized for
  char* pool = nullptr;              // one allocation: 2 in + 2 out chunk SoAs + 3 flux arrays
  grpic_particles in[kBufs], out[kBufs];
  double* flux[3] = {nullptr, nullptr, nullptr};
  int64_t* n_alive_dev = nullptr;    // [kBufs]
  int64_t* n_alive_pin = nullptr;    // pinned host mirror [kBufs]
  uint32_t* status_dev = nullptr;
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
  cudaEvent_t h2d_done[kBufs], push_done[kBufs], d2h_done[kBufs];
  bool events = false;
};

size_t soa_bytes(int64_t n) { return (size_t)n * (7 * sizeof(double) + 2 * sizeof(uint32_t)); }

void carve(char*& p, grpic_particles& q, int64_t n) {
  double** d[7] = {&q.x1, &q.x2, &q.x3, &q.u1, &q.u2, &q.u3, &q.w};
  for (int k = 0; k < 7; ++k) { *d[k] = (double*)p; p += (size_t)n * sizeof(double); }
  q.cell = (uint32_t*)p; p += (size_t)n * sizeof(uint32_t);
  q.flag = (uint32_t*)p; p += (size_t)n * sizeof(uint32_t);
  q.n = n;
}

void release(HostStepState* S) {
  if (!S) return;
  if (S->pool) cudaFree(S->pool);
  if (S->n_alive_pin) cudaFreeHost(S->n_alive_pin);
  if (S->s_h2d) cudaStreamDestroy(S->s_h2d);
  if (S->s_d2h) cudaStreamDestroy(S->s_d2h);
  if (S->events)
    for (int b = 0; b < kBufs; ++b) {
      cudaEventDestroy(S->h2d_done[b]);
      cudaEventDestroy(S->push_done[b]);
      cudaEventDestroy(S->d2h_done[b]);
    }
  delete S;
}

int prepare(grpic_ctx* ctx, int64_t chunk) {
  HostStepState* S = (HostStepState*)ctx->host_step;
  if (S && S->chunk == chunk) return GRPIC_OK;
  release(S);
  ctx->host_step = nullptr;
  S = new (std::nothrow) HostStepState();
  if (!S) return GRPIC_ERR_ALLOC;
  const size_t n2 = ctx->g.size();
  const size_t one = (soa_bytes(chunk) + 255) & ~(size_t)255;
  const size_t total = 2 * kBufs * one + 3 * n2 * sizeof(double) + 256;
  if (cudaMalloc(&S->pool, total) != cudaSuccess) { delete S; return GRPIC_ERR_ALLOC; }
  char* p = S->pool;
  for (int b = 0; b < kBufs; ++b) { char* q = p; carve(q, S->in[b], chunk); p += one; }
  for (int b = 0; b < kBufs; ++b) { char* q = p; carve(q, S->out[b], chunk); p += one; }
  for (int c = 0; c < 3; ++c) { S->flux[c] = (double*)p; p += n2 * sizeof(double); }
  S->n_alive_dev = (int64_t*)p;
  S->status_dev = (uint32_t*)(p + kBufs * sizeof(int64_t));
  bool ok = cudaMallocHost(&S->n_alive_pin, kBufs * sizeof(int64_t)) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&S->s_h2d, cudaStreamNonBlocking) == cudaSuccess;
  ok = ok && cudaStreamCreateWithFlags(&S->s_d2h, cudaStreamNonBlocking) == cudaSuccess;
  if (ok) {
    for (int b = 0; b < kBufs && ok; ++b) {
      ok = cudaEventCreateWithFlags(&S->h2d_done[b], cudaEventDisableTiming) == cudaSuccess &&
           cudaEventCreateWithFlags(&S->push_done[b], cudaEventDisableTiming) == cudaSuccess &&
           cudaEventCreateWithFlags(&S->d2h_done[b], cudaEventDisableTiming) == cudaSuccess;
    }
    S->events = ok;
  }
  if (!ok) { release(S); return GRPIC_ERR_CUDA; }
  S->chunk = chunk;
  ctx->host_step = S;
  return GRPIC_OK;
}

// copy particles [lo, lo+m) of the SoA `src` to [0, m) ... or [dlo, dlo+m) of `dst`
// (the push reads no cell index, so the way in skips it; the way home carries everything)
int copy_soa(const grpic_particles& dst, int64_t dlo, const grpic_particles& src, int64_t slo, int64_t m,
             bool with_cell, cudaMemcpyKind kind, cudaStream_t st) {
  if (m <= 0) return GRPIC_OK;
  double* const d[7] = {dst.x1, dst.x2, dst.x3, dst.u1, dst.u2, dst.u3, dst.w};
  double* const s[7] = {src.x1, src.x2, src.x3, src.u1, src.u2, src.u3, src.w};
  for (int k = 0; k < 7; ++k)
    GRPIC_CUDA_OK(cudaMemcpyAsync(d[k] + dlo, s[k] + slo, (size_t)m * sizeof(double), kind, st));
  if (with_cell)
    GRPIC_CUDA_OK(cudaMemcpyAsync(dst.cell + dlo, src.cell + slo, (size_t)m * sizeof(uint32_t), kind, st));
  GRPIC_CUDA_OK(cudaMemcpyAsync(dst.flag + dlo, src.flag + slo, (size_t)m * sizeof(uint32_t), kind, st));
  return GRPIC_OK;
}

}  // namespace

void grpic_host_step_release(grpic_ctx* ctx) {
  release((HostStepState*)ctx->host_step);
  ctx->host_step = nullptr;
}

extern "C" int grpic_step_host(grpic_ctx* ctx, grpic_particles* host_ptc, grpic_fields* fields,
                               const grpic_fields* background, grpic_current* host_J, double dt,
                               int32_t filter_passes, int64_t chunk_particles, uint32_t* host_status,
                               void* stream) {
  if (!ctx || !host_ptc || !fields || !(dt > 0.0) || host_ptc->n < 0 || filter_passes < 0) return GRPIC_ERR_ARG;
  const int64_t n = host_ptc->n;
  if (n > 0 && (!host_ptc->x1 || !host_ptc->x2 || !host_ptc->x3 || !host_ptc->u1 || !host_ptc->u2 ||
                !host_ptc->u3 || !host_ptc->w || !host_ptc->cell || !host_ptc->flag))
    return GRPIC_ERR_ARG;
  if (host_J && (!host_J->Fr || !host_J->Fth || !host_J->Fph)) return GRPIC_ERR_ARG;
  int64_t chunk = chunk_particles > 0 ? chunk_particles : (int64_t)4 << 20;
  chunk = (chunk + 63) & ~(int64_t)63;               // keeps every SoA member 16-byte aligned
  int rc = prepare(ctx, chunk);
  if (rc != GRPIC_OK) return rc;
  HostStepState* S = (HostStepState*)ctx->host_step;
  cudaStream_t st = (cudaStream_t)stream;
  const size_t n2 = ctx->g.size();
  grpic_current flux = {S->flux[0], S->flux[1], S->flux[2]};
  for (int c = 0; c < 3; ++c) GRPIC_CUDA_OK(cudaMemsetAsync(S->flux[c], 0, n2 * sizeof(double), st));
  GRPIC_CUDA_OK(cudaMemsetAsync(S->status_dev, 0, sizeof(uint32_t), st));

  // an error return must not leave copies into the caller's host memory in flight
  auto fail = [&](int code) -> int {
    cudaStreamSynchronize(S->s_h2d);
    cudaStreamSynchronize(S->s_d2h);
    cudaStreamSynchronize(st);
    return code;
  };
  const int64_t nchunks = (n + chunk - 1) / chunk;
  int64_t written = 0;                                // survivors copied back so far
  auto finish = [&](int64_t c) -> int {               // chunk c: count known -> copy survivors home
    const int b = (int)(c % kBufs);
    GRPIC_CUDA_OK(cudaEventSynchronize(S->push_done[b]));
    const int64_t m = S->n_alive_pin[b];
    GRPIC_CUDA_OK(cudaStreamWaitEvent(S->s_d2h, S->push_done[b], 0));
    int r = copy_soa(*host_ptc, written, S->out[b], 0, m, true, cudaMemcpyDeviceToHost, S->s_d2h);
    if (r != GRPIC_OK) return r;
    GRPIC_CUDA_OK(cudaEventRecord(S->d2h_done[b], S->s_d2h));
    written += m;
    return GRPIC_OK;
  };
  for (int64_t c = 0; c < nchunks; ++c) {
    const int b = (int)(c % kBufs);
    const int64_t lo = c * chunk, m = (n - lo < chunk) ? n - lo : chunk;
    // input buffer b is free once the push of chunk c-2 has read it
    if (c >= kBufs) GRPIC_CUDA_OK(cudaStreamWaitEvent(S->s_h2d, S->push_done[b], 0));
    rc = copy_soa(S->in[b], 0, *host_ptc, lo, m, false, cudaMemcpyHostToDevice, S->s_h2d);
    if (rc != GRPIC_OK) return fail(rc);
    GRPIC_CUDA_OK(cudaEventRecord(S->h2d_done[b], S->s_h2d));
    GRPIC_CUDA_OK(cudaStreamWaitEvent(st, S->h2d_done[b], 0));
    if (c >= kBufs) GRPIC_CUDA_OK(cudaStreamWaitEvent(st, S->d2h_done[b], 0));   // output buffer b drained
    grpic_particles in = S->in[b], out = S->out[b];
    in.n = m;
    out.n = m;
    rc = grpic_push_deposit_compact(ctx, &in, &out, fields, &flux, dt, S->n_alive_dev + b, S->status_dev, st);
    if (rc != GRPIC_OK) return fail(rc);
    GRPIC_CUDA_OK(cudaMemcpyAsync(S->n_alive_pin + b, S->n_alive_dev + b, sizeof(int64_t),
                                  cudaMemcpyDeviceToHost, st));
    GRPIC_CUDA_OK(cudaEventRecord(S->push_done[b], st));
    if (c >= 1) { rc = finish(c - 1); if (rc != GRPIC_OK) return fail(rc); }
  }
  if (nchunks >= 1) { rc = finish(nchunks - 1); if (rc != GRPIC_OK) return fail(rc); }

  // multi-GPU: sum the fluxes of the ranks' particle shards (one collective on the caller's stream)
  if (ctx->flux_exchange && ctx->flux_exchange(ctx->flux_exchange_user, S->flux[0], 3 * n2, stream) != 0)
    return fail(GRPIC_ERR_CUDA);
  // grid part of the step on the caller's stream, overlapping the last copies home
  rc = grpic_finalize_current(ctx, &flux, filter_passes, st);
  if (rc != GRPIC_OK) return fail(rc);
  rc = grpic_field_step(ctx, fields, &flux, background, dt, st);
  if (rc != GRPIC_OK) return fail(rc);
  if (host_J) {
    double* const hj[3] = {host_J->Fr, host_J->Fth, host_J->Fph};
    for (int c = 0; c < 3; ++c)
      GRPIC_CUDA_OK(cudaMemcpyAsync(hj[c], S->flux[c], n2 * sizeof(double), cudaMemcpyDeviceToHost, st));
  }
  if (host_status)
    GRPIC_CUDA_OK(cudaMemcpyAsync(host_status, S->status_dev, sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
  GRPIC_CUDA_OK(cudaStreamSynchronize(S->s_d2h));
  GRPIC_CUDA_OK(cudaStreamSynchronize(st));
  host_ptc->n = written;                              // survivors, in order, at the front
  return GRPIC_OK;
}
