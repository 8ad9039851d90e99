// types.h — plain structs shared by the host side (plan, C ABI) and the kernels.
#pragma once

namespace galb {

struct SweepParams {
    const void* I;      // profile, T[nr]
    int nr;
    double Rmin, dR, Rmax, dxy, inc_cos;
    double r_dR, r_inc;      // RN(1 / dR), RN(1 / inc_cos) for the exact-division shortcut
    int true_div;            // 1: a reciprocal is not usable (host check), take true divisions
};

// Scalars of one call that the index arithmetic needs (host-computed).  They sit
// in the kernel parameter block so the compiler reads them as constant-bank operands, not registers.
struct IndexScalars {
    double du, rdu;        // du = 1/(N dxy); rdu = RN(1/du) for the exact-division shortcut
    double cos_PA, sin_PA;
    double fH, fHm1, fN1;  // N/2, N/2 - 1, N - 1 as doubles
    int du_exact_div;      // 1: rdu is not usable, take a true division
};

// Per-call scalars (host-computed).
struct CallScalars {
    IndexScalars ix;
    double dRA_turns, dDec_turns;
    int has_phase;
    double amp = 1.0;      // factor on the visibilities and accumulate-into-vis flag: multi-source composition only
    int accumulate = 0;
};

// One placement of a multi-source call: rotation, offsets in turns (rotated), flux factor.
struct Placement {
    double cos_PA, sin_PA, dRA_turns, dDec_turns, amp;
    int has_phase, pad;
};
constexpr int GAL_MULTI_CHUNK = 16;          // placements per launch (they travel in the kernel parameter block)
struct PlacementSet {
    Placement pl[GAL_MULTI_CHUNK];
    int S;
    int init_from_vis;                       // start from the sum already in vis (later chunks of a long list)
};

}  // namespace galb
