// Host planner of the matched-filter search (no CUDA in this file).
//
// The filter of PAPER.md:L106 ("convolving the line of the trajectory with the pixel response
// function") is separable per frame: its x part depends only on the trajectory's x-motion
// (vx, ax), its y part only on (vy, ay).  The planner groups trajectories into AXIS CLASSES
// (distinct x-motions, distinct y-motions) and packs them into BATCHES that share one x-class,
// so that the x-pass of the separable kernel is computed once per batch.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/tno_mf.h"

namespace tno {

// floor(d + 1/2) of d = (v*dt + (a*dt)*dt) + j, all in IEEE double without contraction
// (BASELINE.json:north_star "5x5 window at round(c_t)"; reading c1 in DESIGN.md: ties go up).
// Returns false if the shift does not fit comfortably in 32 bits.
bool axis_shift(double v, double a, double dt, double j, int32_t *shift, bool *tie = nullptr);

struct AxisClass {
    float v, a;                  // px/frame, px/frame^2 (exact float32 values of the ABI)
    int32_t smin, smax;          // extreme integer shifts over t = 0..T-1
    std::vector<int32_t> shift;  // [T]
    bool tie = false;            // some frame has d + 1/2 exactly integer (the rounding is then not odd in d)
    bool jittered = false;       // a non-zero jitter enters the displacement of this class
};

struct Batch {
    int32_t xcls;                // x-class shared by every entry
    std::vector<int32_t> traj;   // trajectory index of each entry (size <= max_entries)
    int32_t max_spread;          // max over t of (max_e sy - min_e sy)
};

// A SLOT of the separable kernel holds the y-motion (v, a) and, when the filter is symmetric under the
// reflection y -> -y, also its mirror image (-v, -a): shift_t and phase_t change sign, the 5 taps reverse,
// so that with the even and odd parts of the taps
//     N_plus  = E + O,   N_minus = E - O,    E = w2 X0 + s1 (X+1 + X-1) + s2 (X+2 + X-2),
//                                            O =         d1 (X+1 - X-1) + d2 (X+2 - X-2)
// both members are accumulated with 5 multiply-adds per pixel and frame instead of 10 (exact algebra;
// DESIGN.md "mirror pairs").  member[0] moves as (v, a) with v > 0 or (v == 0, a >= 0) when the class is
// pairable, member[1] as (-v, -a); either may be absent (-1).  A class that is not pairable (exact rounding
// ties, jitter on the y axis, a filter without the symmetry) sits alone in member[0] in its own orientation.
struct Slot {
    int32_t member[2];           // trajectory indices or -1
    int32_t ycls;                // y-class the tables are built from (index into Plan::ycls)
    int32_t flip;                // 1: that class is the mirror image of the slot's orientation
};

struct SlotBatch {
    int32_t xcls;
    std::vector<Slot> slots;     // size <= max_slots
};

struct Plan {
    int32_t T = 0;
    double t0 = 0.0;
    std::vector<AxisClass> xcls, ycls;
    std::vector<int32_t> traj_xc, traj_yc;   // [n_traj]
    std::vector<Batch> batches;
    std::vector<SlotBatch> slot_batches;
};

// Group trajectories into axis classes.  Returns TNO_MF_OK or TNO_MF_EINVAL (shift overflow).
// frame_times (HOST [T], NULL = the frame index) and jitter_xy (HOST [T][2] px, NULL = none) enter the
// displacement of every class: c_t = (x, y) + v (tau_t - t0) + a (tau_t - t0)^2 + j_t.
int build_classes(const tno_mf_traj *traj, int32_t n_traj, int32_t T, double t0, const float *frame_times,
                  const float *jitter_xy, Plan *plan);

// Pack the trajectories of each x-class into batches of at most max_entries entries whose integer
// y-shifts never differ by more than max_spread in any frame.  Entries are ordered by (vy, ay) so
// that neighbours move alike.  A single trajectory always fits (spread 0).
// max_spread >= kUnlimitedSpread (what the search itself uses): no spread limit, and each x-class
// is split into the fewest batches, of sizes that differ by at most one.
constexpr int32_t kUnlimitedSpread = 1 << 30;
void build_batches(Plan *plan, int32_t max_entries, int32_t max_spread);

// Pack the trajectories of each x-class into slots (mirror pairs where `symmetric_filter` and the class
// allow it) and the slots, ordered by (|v|-orientation v, a), into the fewest batches of at most max_slots
// slots, of sizes that differ by at most one.  Duplicate trajectories get slots of their own.
void build_slot_batches(Plan *plan, int32_t max_slots, bool symmetric_filter);

}  // namespace tno
