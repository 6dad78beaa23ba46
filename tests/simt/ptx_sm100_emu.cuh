// ptx_sm100_emu.cuh — TEST INFRASTRUCTURE (see simt_shim.h).  Host stand-ins for the inline-PTX helpers of
// paper_2606_14603_b200/csrc/ptx_sm100.cuh, with the semantics the PTX ISA gives them: an mbarrier has an arrival
// count and a transaction-byte count; a phase completes when both reach zero, which flips the phase bit and re-arms the
// arrival count; try_wait.parity(P) is true once the phase with parity P has completed.  A bulk copy moves its bytes
// and credits them to the barrier; its operands must be 16-byte aligned and the size a multiple of 16 (checked).
// tests/simt/build.py installs this file as "ptx_sm100.cuh" of the emulation build.
#pragma once
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>

// The barrier words themselves are touched by many fibres between rendezvous: not data, so not for ThreadSanitizer.
#define EMU_BAR __attribute__((no_sanitize("thread")))

namespace molsim {

struct EmuMbar { uint32_t phase : 1, pending : 15, count : 16; int32_t tx; };
static_assert(sizeof(EmuMbar) == 8, "an mbarrier is one 64-bit shared-memory word");

EMU_BAR inline EmuMbar* emu_bar(unsigned long long* bar) { return reinterpret_cast<EmuMbar*>(bar); }
EMU_BAR inline void emu_bar_settle(EmuMbar* m) {
  if (m->pending == 0 && m->tx == 0) { m->phase ^= 1u; m->pending = m->count; }
  simt::note_progress();
}
inline void emu_fail(const char* what) { std::fprintf(stderr, "simt ptx: %s\n", what); std::abort(); }

EMU_BAR inline void mbar_init(unsigned long long* bar, uint32_t count) {
  EmuMbar* m = emu_bar(bar);
  m->phase = 0; m->pending = count; m->count = count; m->tx = 0;
}
inline void fence_mbar_init() {}
EMU_BAR inline void mbar_expect_tx(unsigned long long* bar, uint32_t bytes) {
  EmuMbar* m = emu_bar(bar);
  simt::hb_release(bar);
  if (m->pending == 0) emu_fail("mbarrier arrival beyond the expected count");
  m->tx += (int32_t)bytes; m->pending--;
  emu_bar_settle(m);
}
EMU_BAR inline void mbar_arrive(unsigned long long* bar) {
  EmuMbar* m = emu_bar(bar);
  simt::hb_release(bar);                 // what this thread did before arriving is visible to whoever waits the phase out
  if (m->pending == 0) emu_fail("mbarrier arrival beyond the expected count");
  m->pending--;
  emu_bar_settle(m);
}
EMU_BAR inline bool mbar_try_wait(unsigned long long* bar, uint32_t parity) {
  if (emu_bar(bar)->phase != (parity & 1u)) { simt::hb_acquire(bar); return true; }
  simt::run_deferred(bar);               // adversarial mode: a copy lands no earlier than the first poll that waits for it
  simt::yield();                         // the callers spin on this
  return false;
}
inline void fence_proxy_async() {}
EMU_BAR inline void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* bar) {
  if (((uintptr_t)dst | (uintptr_t)src | bytes) & 15u) emu_fail("bulk copy operands must be 16-byte aligned multiples of 16");
  auto land = [=]() EMU_BAR {
    simt::hb_acquire(bar);                 // the copy was issued after the issuer's expect_tx on this barrier: a late landing
                                           // (seeded schedules: done by whichever fibre polls first) keeps that order
    std::memcpy(dst, src, bytes);          // the async proxy's write
    simt::hb_release(bar);
    EmuMbar* m = emu_bar(bar);
    m->tx -= (int32_t)bytes;
    emu_bar_settle(m);
  };
  if (!simt::defer(bar, land)) land();
}
inline void prefetch_l1(const void* ptr) {
  (void)*reinterpret_cast<const volatile unsigned char*>(ptr);     // a prefetch of an unmapped address is dropped on the
}                                                                  // GPU; here it must at least lie inside an allocation

}  // namespace molsim
