// device_common.cuh - device helpers shared by kernels.cu and group_kernel.cu: HH rate functions,
// bulk-async copy (TMA) / mbarrier primitives, the per-cell runtime of a (sub-)step.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

namespace arbb {
namespace {

constexpr unsigned kFull = 0xffffffffu;

// ------------------------------------------------------------------------------------------
// HH rate functions (reading R5): textbook Hodgkin-Huxley 1952, 6.3 C, rest at -65 mV.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ double exprelr(double x) { return x == 0.0 ? 1.0 : x / expm1(x); }

struct Rates { double am, bm, ah, bh, an, bn; };
__device__ __forceinline__ Rates hh_rates(double v) {
  Rates r;
  r.am = exprelr(-(v + 40.0) / 10.0);
  r.bm = 4.0 * exp(-(v + 65.0) / 18.0);
  r.ah = 0.07 * exp(-(v + 65.0) / 20.0);
  r.bh = 1.0 / (1.0 + exp(-(v + 35.0) / 10.0));
  r.an = 0.1 * exprelr(-(v + 55.0) / 10.0);
  r.bn = 0.125 * exp(-(v + 65.0) / 80.0);
  return r;
}

// ------------------------------------------------------------------------------------------
// bulk-async copy (TMA) and mbarrier primitives
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t addr = smem_u32(bar);
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(addr), "r"(parity)
        : "memory");
  } while (!ok);
}

// shared -> global bulk copy (TMA store) and its completion
__device__ __forceinline__ void bulk_s2g(void* dst_gmem, const void* src_smem, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst_gmem), "r"(smem_u32(src_smem)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// ask the TMA unit to bring a range into L2 (no destination in shared memory)
__device__ __forceinline__ void bulk_prefetch_l2(const void* src_gmem, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}

// per-cell runtime of the (sub-)step in progress, in shared memory
struct CellS {
  double *tcur, *tnext, *delta, *vprev;
  uint32_t *evcur, *evend, *armed, *mode, *wb, *dirty;
};
__device__ __forceinline__ CellS carve_cells(uint8_t* p, uint32_t cap) {
  CellS c;
  c.tcur = (double*)p; c.tnext = c.tcur + cap; c.delta = c.tnext + cap; c.vprev = c.delta + cap;
  c.evcur = (uint32_t*)(c.vprev + cap); c.evend = c.evcur + cap; c.armed = c.evend + cap;
  c.mode = c.armed + cap; c.wb = c.mode + cap; c.dirty = c.wb + cap;
  return c;
}


}  // namespace
}  // namespace arbb
