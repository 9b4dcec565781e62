// toggles.h - the environment toggles of libpulse.so (listed in include/pulse.h), read ONCE per process at first use.
// None changes results beyond the order of fp32 sums; they exist to cross-check one kernel against another.
#pragma once
#include <cstdlib>

namespace pulse {

struct Toggles {
  bool no_pdl;            // PULSE_NO_PDL=1          ordinary stream-ordered launches (no programmatic dependent launch)
  bool no_side_stream;    // PULSE_NO_SIDE_STREAM=1  everything on the caller's stream
  bool no_gn_fused;       // PULSE_NO_GN_FUSED=1     GroupNorm backward always as two kernels (= PULSE_FLAG_GN_TWO_PASS)
  bool conv_1cta;         // PULSE_CONV_1CTA=1       single-CTA tcgen05 conv kernel everywhere (= PULSE_FLAG_CONV_1CTA)
  bool wgrad_1cta;        // PULSE_WGRAD_1CTA=1      single-CTA tcgen05 wgrad kernel everywhere
  bool no_split_k;        // PULSE_NO_SPLIT_K=1      no cluster split-K in the pair conv kernel (few-tile convs then take the single-CTA kernel)
  int conv_1cta_tiles;    // PULSE_CONV_1CTA_TILES=k convs with <= k single-CTA tiles take the single-CTA kernel (-1: default)
};

inline const Toggles& toggles() {
  static const Toggles t = [] {
    auto on = [](const char* name) { const char* e = getenv(name); return e && e[0] == '1'; };
    Toggles v;
    v.no_pdl = on("PULSE_NO_PDL"); v.no_side_stream = on("PULSE_NO_SIDE_STREAM"); v.no_gn_fused = on("PULSE_NO_GN_FUSED");
    v.conv_1cta = on("PULSE_CONV_1CTA"); v.wgrad_1cta = on("PULSE_WGRAD_1CTA"); v.no_split_k = on("PULSE_NO_SPLIT_K");
    const char* e = getenv("PULSE_CONV_1CTA_TILES");
    v.conv_1cta_tiles = e ? atoi(e) : -1;
    return v;
  }();
  return t;
}

}  // namespace pulse
