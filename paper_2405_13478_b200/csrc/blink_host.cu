// blink_host.cu -- blink_grid_image_host: the end-to-end form of blink_grid_image for data that lives
// in HOST memory.  The paper keeps everything on the device ("process the data fully inside GPU
// memory") and lists the interleaving of "kernel executions on portions of data ... with
// memory transfers" and pinned host memory as its next optimisation; this is that:
// the batch is cut into chunks of time steps, and the host-to-device copy of chunk i + 1, the imaging
// of chunk i and the device-to-host copy of chunk i - 1 run concurrently on three streams over a ring
// of plan-owned staging buffers.  Pure plumbing around blink_grid_image: every step of the path still
// runs in the kernels of blink_fused.cu / blink_image*.cu.
#include <algorithm>
#include <vector>

#include "blink_internal.h"

namespace blink {

void host_pipe_free(blink_plan *p) {
  HostPipe &h = p->hp;
  for (int b = 0; b < HostPipe::kDepth; ++b) {
    cudaFree(h.d_vis[b]);
    cudaFree(h.d_img[b]);
    if (h.in_done[b]) cudaEventDestroy(h.in_done[b]);
    if (h.cmp_done[b]) cudaEventDestroy(h.cmp_done[b]);
    if (h.out_done[b]) cudaEventDestroy(h.out_done[b]);
  }
  if (h.start) cudaEventDestroy(h.start);
  for (int s = 0; s < 3; ++s) {
    if (h.done[s]) cudaEventDestroy(h.done[s]);
    if (h.st[s]) cudaStreamDestroy(h.st[s]);
  }
  h = HostPipe();
}

}  // namespace blink

using namespace blink;

extern "C" int blink_plan_reserve_host(blink_plan *p, int chunk_t) {
  if (!p || chunk_t < 0) return BLINK_EINVAL;
  int rc = check_device(p);
  if (rc != BLINK_OK) return rc;
  HostPipe &h = p->hp;
  if (chunk_t == 0) {
    // auto: about 32 MiB each way per chunk -- small enough that filling and draining the three-stage pipeline is
    // a few per cent of a batch, large enough for the copies to run at the link rate (measured on the station,
    // 0.84 GB each way per step: 1 step per chunk 20.0 ms, 4 steps = 33 MB 18.1 ms, 13 steps 18.9 ms, 50 steps 24.1 ms)
    if (h.chunk_t > 0) return BLINK_OK;
    const size_t per_t = std::max(sizeof(float2) * (size_t)p->n_ch * p->n_bl, sizeof(float) * (size_t)p->n_ch * p->n_pix * p->n_pix);
    chunk_t = (int)std::max<size_t>(1, (((size_t)32 << 20) + per_t / 2) / per_t);
  }
  if (chunk_t <= h.chunk_t) return BLINK_OK;
  BLINK_CUDA_TRY(cudaDeviceSynchronize(), "blink_plan_reserve_host sync");
  host_pipe_free(p);
  rc = image_reserve(p, chunk_t);                 // blink_grid_image's own scratch for a chunk
  if (rc != BLINK_OK) return rc;
  const size_t vb = sizeof(float2) * (size_t)chunk_t * p->n_ch * p->n_bl;
  const size_t ib = sizeof(float) * (size_t)chunk_t * p->n_ch * p->n_pix * p->n_pix;
  cudaError_t e = cudaSuccess;
  auto step = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
  for (int b = 0; b < HostPipe::kDepth; ++b) {
    step(cudaMalloc((void **)&h.d_vis[b], vb));
    step(cudaMalloc((void **)&h.d_img[b], ib));
    step(cudaEventCreateWithFlags(&h.in_done[b], cudaEventDisableTiming));
    step(cudaEventCreateWithFlags(&h.cmp_done[b], cudaEventDisableTiming));
    step(cudaEventCreateWithFlags(&h.out_done[b], cudaEventDisableTiming));
  }
  step(cudaEventCreateWithFlags(&h.start, cudaEventDisableTiming));
  for (int s = 0; s < 3; ++s) {
    step(cudaStreamCreateWithFlags(&h.st[s], cudaStreamNonBlocking));
    step(cudaEventCreateWithFlags(&h.done[s], cudaEventDisableTiming));
  }
  if (e != cudaSuccess) {
    set_cuda_error(e, "blink_plan_reserve_host");
    host_pipe_free(p);
    return e == cudaErrorMemoryAllocation ? BLINK_ENOMEM : BLINK_ECUDA;
  }
  h.chunk_t = chunk_t;
  return BLINK_OK;
}

extern "C" int blink_grid_image_host(blink_plan *p, const void *vis_host, int n_t, void *images_host, void *stream) {
  if (!p || n_t < 0) return BLINK_EINVAL;
  if (n_t == 0) return BLINK_OK;
  if (!vis_host || !images_host) return BLINK_EINVAL;
  int rc = check_device(p);
  if (rc == BLINK_OK) rc = check_corrections_current(p);
  if (rc != BLINK_OK) return rc;
  HostPipe &h = p->hp;
  if (h.chunk_t < 1) return BLINK_ERESERVE;
  cudaStream_t cur = (cudaStream_t)stream;
  cudaStream_t s_in = h.st[0], s_cmp = h.st[1], s_out = h.st[2];
  const size_t v_t = sizeof(float2) * (size_t)p->n_ch * p->n_bl;             // bytes per time step
  const size_t i_t = sizeof(float) * (size_t)p->n_ch * p->n_pix * p->n_pix;
  const unsigned char *vh = (const unsigned char *)vis_host;
  unsigned char *ih = (unsigned char *)images_host;
  cudaError_t e = cudaSuccess;
  auto step = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
  // everything below is ordered after what `stream` holds now
  step(cudaEventRecord(h.start, cur));
  for (int s = 0; s < 3; ++s) step(cudaStreamWaitEvent(h.st[s], h.start, 0));
  // chunk sizes: 1, 2, 4, ... up to chunk_t at the start and back down at the end, so that the first copy in and
  // the last copy out -- the part of the batch during which only one direction of the link is busy -- are short
  std::vector<int> ks;
  {
    int ramp = 0;
    for (int k = 1; k < h.chunk_t; k *= 2) ramp += k;
    int rem = n_t;
    if (2 * ramp + h.chunk_t <= n_t) {
      for (int k = 1; k < h.chunk_t; k *= 2) ks.push_back(k);
      rem -= 2 * ramp;
    }
    const size_t n_up = ks.size();
    for (; rem > 0; rem -= h.chunk_t) ks.push_back(std::min(h.chunk_t, rem));
    for (size_t j = n_up; j-- > 0;) ks.push_back(ks[j]);
  }
  int i = 0, t0 = 0;
  for (; i < (int)ks.size() && e == cudaSuccess; t0 += ks[i], ++i) {
    const int k = ks[i], b = i % HostPipe::kDepth;
    if (i >= HostPipe::kDepth) step(cudaStreamWaitEvent(s_in, h.cmp_done[b], 0));      // d_vis[b] has been consumed
    step(cudaMemcpyAsync(h.d_vis[b], vh + (size_t)t0 * v_t, (size_t)k * v_t, cudaMemcpyHostToDevice, s_in));
    step(cudaEventRecord(h.in_done[b], s_in));
    step(cudaStreamWaitEvent(s_cmp, h.in_done[b], 0));
    if (i >= HostPipe::kDepth) step(cudaStreamWaitEvent(s_cmp, h.out_done[b], 0));     // d_img[b] has been copied out
    if (e != cudaSuccess) break;
    rc = blink_grid_image(p, h.d_vis[b], k, h.d_img[b], (void *)s_cmp);
    if (rc != BLINK_OK) break;
    step(cudaEventRecord(h.cmp_done[b], s_cmp));
    step(cudaStreamWaitEvent(s_out, h.cmp_done[b], 0));
    step(cudaMemcpyAsync(ih + (size_t)t0 * i_t, h.d_img[b], (size_t)k * i_t, cudaMemcpyDeviceToHost, s_out));
    step(cudaEventRecord(h.out_done[b], s_out));
  }
  // `stream` continues when all three are done (also on the error path, so nothing is left dangling)
  for (int s = 0; s < 3; ++s) {
    cudaEventRecord(h.done[s], h.st[s]);
    cudaStreamWaitEvent(cur, h.done[s], 0);
  }
  if (rc != BLINK_OK) return rc;
  if (e != cudaSuccess) {
    set_cuda_error(e, "blink_grid_image_host");
    return BLINK_ECUDA;
  }
  return BLINK_OK;
}
