// stream_probe.cuh -- read-only HBM streaming ceilings, measured by bench.py in the same run as the
// draft step ("a read-only streaming-sum microbenchmark measured in the same run as the
// practical ceiling"). No arithmetic of the method lives here. Two probes over the same buffer:
//   k_stream_sum   classic: every thread sums 16-byte loads, grid-stride, 8 loads in flight per thread;
//   k_stream_bulk  the GEMV's own data path without its arithmetic: one CTA per SM, producer warps issue
//                  1-D bulk async copies (cp.async.bulk, SASS UBLKCP) of `seg` bytes into a shared-memory
//                  ring guarded by full / empty mbarriers, the consumer warp releases each stage at once.
// Both read `bytes` bytes exactly once; the host divides by the kernel's duration.
#pragma once
#include "ptx.cuh"

namespace dvt {

__global__ void __launch_bounds__(512) k_stream_sum(const uint4* __restrict__ buf, int64_t n16, float* sink) {
  const int64_t stride = static_cast<int64_t>(gridDim.x) * blockDim.x;
  int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  uint32_t acc = 0;
  for (; i + 7 * stride < n16; i += 8 * stride) {
    uint4 v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = __ldcs(buf + i + j * stride);
#pragma unroll
    for (int j = 0; j < 8; ++j) acc += v[j].x ^ v[j].y ^ v[j].z ^ v[j].w;
  }
  for (; i < n16; i += stride) {
    const uint4 v = __ldcs(buf + i);
    acc += v.x ^ v.y ^ v.z ^ v.w;
  }
  if (acc == 0x9e3779b9u) *sink = 1.f;  // keeps the loads alive; practically never true
}

constexpr int kProbeProducerWarps = 4;
constexpr int kProbeThreads = 32 * (kProbeProducerWarps + 1);

// grid = number of SMs; CTA c reads the contiguous range [c, c + 1) * bytes / grid (16-byte aligned) in
// stages of `rows` segments of `seg` bytes; ring of n_stages stages.
__global__ void __launch_bounds__(kProbeThreads, 1) k_stream_bulk(const uint8_t* __restrict__ buf, int64_t bytes, int seg,
                                                                  int rows, int n_stages, float* sink) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int stage_bytes = rows * seg;
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + static_cast<size_t>(n_stages) * stage_bytes);
  uint64_t* empty = full + 8;
  const int64_t per = (bytes / gridDim.x) & ~static_cast<int64_t>(15);
  const uint8_t* src = buf + per * blockIdx.x;
  const int64_t n_seg = per / seg;                       // whole segments of this CTA (the tail is dropped: < seg bytes)
  const int64_t n_st = (n_seg + rows - 1) / rows;
  if (tid == 0) {
    for (int s = 0; s < n_stages; ++s) {
      mbar_init(&full[s], kProbeProducerWarps);
      mbar_init(&empty[s], 1);
    }
    mbar_fence_init();
  }
  __syncthreads();
  if (warp < kProbeProducerWarps) {
    const uint64_t pol = l2_policy_evict_first();
    const int rpw = (rows + kProbeProducerWarps - 1) / kProbeProducerWarps;  // segments per producer warp, <= 32
    int slot = 0, round = 0;
    for (int64_t s = 0; s < n_st; ++s) {
      if (round > 0) mbar_wait(&empty[slot], (round & 1) ^ 1);
      const int64_t seg0 = s * rows + warp * rpw;
      const int mine = static_cast<int>(max(static_cast<int64_t>(0), min(static_cast<int64_t>(rpw), min(static_cast<int64_t>(rows - warp * rpw), n_seg - seg0))));
      if (lane == 0) mbar_arrive_expect_tx(&full[slot], static_cast<uint32_t>(mine) * seg);
      __syncwarp();
      if (lane < mine)
        bulk_g2s(smem + static_cast<size_t>(slot) * stage_bytes + static_cast<size_t>(warp * rpw + lane) * seg,
                 src + (seg0 + lane) * seg, seg, &full[slot], pol);
      if (++slot == n_stages) { slot = 0; ++round; }
    }
    return;
  }
  // consumer warp: a stage is released as soon as it has landed
  uint32_t acc = 0;
  int slot = 0, round = 0;
  for (int64_t s = 0; s < n_st; ++s) {
    mbar_wait(&full[slot], round & 1);
    acc += reinterpret_cast<const uint32_t*>(smem + static_cast<size_t>(slot) * stage_bytes)[lane];
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[slot]);
    if (++slot == n_stages) { slot = 0; ++round; }
  }
  if (acc == 0x9e3779b9u) *sink = 1.f;
}

}  // namespace dvt
