// sla_tc_common.cuh -- the streamed-ring machinery of the warp-per-head kernels (forward `sla_fwd_tc.cu`, backward
// `sla_bwd_tc.cu`) on top of sla_tc_base.cuh: the per-warp consumer view of a TMA ring and its addressing.
//
// Include it INSIDE the translation unit's `namespace sla { namespace { ... } }`, after defining
//   constexpr int NST  (ring stages per stream)  and  template <int D> struct Cfg { SR, BOX_BYTES, ... }.
#ifndef SLA_TC_COMMON_INCLUDED
#define SLA_TC_COMMON_INCLUDED

#include "sla_tc_base.cuh"

// ---- per-warp consumer view of one ring -----------------------------------------------------------
// Stage st of a stream holds rows [R0 + st*SR, R0 + (st+1)*SR).  `waited` = stages whose full barrier
// this warp has observed; `released` = stages this warp has handed back to the producer.  The ring slot
// and barrier phase of the next stage to wait for / to release are tracked incrementally (no division
// by the stage count in the hot loops): stage st lives in slot (st + bias) mod NST for every stage that
// has not been released yet, with bias = r_slot - released.
struct RingView {
  uint32_t base;      // shared address of slot 0
  uint32_t full;      // shared address of full barriers [NST]
  uint32_t empty;     // shared address of empty barriers [NST]
  int waited;
  int released;
  int w_slot, w_phase;   // slot and parity of stage `waited`
  int r_slot, bias;      // slot of stage `released`; bias = r_slot - released
  int nst;               // stages of this ring (a compile-time constant of the caller: folds after inlining)
};
__device__ __forceinline__ RingView make_ring(uint32_t base, uint32_t full, uint32_t empty, int nst = NST) {
  return RingView{base, full, empty, 0, 0, 0, 0, 0, 0, nst};
}

__device__ __forceinline__ void ring_wait_upto(RingView& rv, int stage_last) {
  while (rv.waited <= stage_last) {
    mbar_wait(rv.full + 8u * rv.w_slot, (uint32_t)rv.w_phase);
    ++rv.waited;
    if (++rv.w_slot == rv.nst) { rv.w_slot = 0; rv.w_phase ^= 1; }
  }
}
// Release every stage that lies entirely below relative row `rel` (rows are relative to R0).
template <int SR>
__device__ __forceinline__ void ring_release_below(RingView& rv, int rel) {
  while ((rv.released + 1) * SR <= rel) {
    ring_wait_upto(rv, rv.released);   // never release a stage before it has landed (phase pacing)
    __syncwarp();
    if ((threadIdx.x & 31) == 0) mbar_arrive(rv.empty + 8u * rv.r_slot);
    ++rv.released;
    if (++rv.r_slot == rv.nst) { rv.r_slot = 0; rv.bias -= rv.nst; }
  }
}
// Steady state of a loop whose step is exactly one stage of rows: after the first step of a pass,
// every further step starts SR rows later, so exactly one more stage -- the oldest unreleased one, which
// the previous step has read and therefore waited for -- lies entirely below it.
__device__ __forceinline__ void ring_release_one(RingView& rv) {
  __syncwarp();
  if ((threadIdx.x & 31) == 0) mbar_arrive(rv.empty + 8u * rv.r_slot);
  ++rv.released;
  if (++rv.r_slot == rv.nst) { rv.r_slot = 0; rv.bias -= rv.nst; }
}

// Shared address of (relative row rel, 16-byte chunk `chunk` of this slab row) inside a ring whose
// slots are `slot_bytes` apart; the tensor's stage starts `toff` bytes into the slot.  The row must
// belong to a stage that has been waited for and not yet released.
template <int D>
__device__ __forceinline__ uint32_t ring_addr(const RingView& rv, int slot_bytes, int toff, int rel, int chunk) {
  using C = Cfg<D>;
  const int st = (int)((unsigned)rel / (unsigned)C::SR), r = (int)((unsigned)rel % (unsigned)C::SR);   // rel >= 0
  int slot = st + rv.bias;
  if (slot >= rv.nst) slot -= rv.nst;
  const int box = chunk >> 3, cib = chunk & 7;
  return rv.base + (uint32_t)(slot * slot_bytes + toff + box * C::BOX_BYTES + r * 128 +
                              ((cib ^ (r & 7)) << 4));
}

#endif  // SLA_TC_COMMON_INCLUDED
