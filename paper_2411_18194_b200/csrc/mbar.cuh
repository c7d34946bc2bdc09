// mbar.cuh -- the slow side of an mbarrier wait, shared by the TMA kernels (demag_tile.cu, local.cu).
//
// A wait first polls mbarrier.try_wait in the kernel itself (the copy normally lands within a few polls).  Only when
// 65 536 polls have failed does it come here: poll with a __nanosleep back-off and give up by wall time, not by poll
// count.  A copy that is merely slow -- ncu replay, MPS or time-slicing, a debugger, eight worlds sharing the GPU -- is
// waited for; only a copy that has not landed after MMX_MBAR_TIMEOUT_NS (10 s on %globaltimer) is taken for a lost one,
// and the kernel traps rather than hang the GPU for good (the host then sees a CUDA error from the next call).
#pragma once

#ifndef MMX_MBAR_TIMEOUT_NS
#define MMX_MBAR_TIMEOUT_NS 10000000000ull
#endif

static __device__ __noinline__ void mmx_mbar_wait_slow(unsigned bar_s32, unsigned parity) {
  unsigned long long t0, t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
  unsigned ok = 0, ns = 64;
  while (true) {
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(ok) : "r"(bar_s32), "r"(parity) : "memory");
    if (ok) return;
    __nanosleep(ns);
    if (ns < 4096) ns *= 2;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    if (t - t0 > MMX_MBAR_TIMEOUT_NS) __trap();
  }
}
