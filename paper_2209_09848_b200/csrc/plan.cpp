// Host planner: axis classes and batches (see plan.h).  Compiled with -ffp-contract=off so that
// the displacement is evaluated exactly as on the device (separately rounded mul/add).
#include "plan.h"

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <map>
#include <utility>

namespace tno {

bool axis_shift(double v, double a, double dt, double j, int32_t *shift, bool *tie) {
    volatile double p1 = v * dt;          // volatile: keep the operations separately rounded, in the
    volatile double adt = a * dt;         // order the device (tables.cu) and the oracle use
    volatile double p2 = adt * dt;
    volatile double d0 = p1 + p2;
    const double d = d0 + j;
    const double f = std::floor(d + 0.5);
    if (!(std::fabs(f) < 1.0e9)) return false;
    // d + 1/2 is exact for |d| < 2^51, so this is the exact tie test (floor(-d + 1/2) != -floor(d + 1/2))
    if (tie) *tie = (d + 0.5 == f);
    *shift = (int32_t)f;
    return true;
}

static uint64_t key_of(float v, float a) {
    uint32_t bv, ba;
    v += 0.0f; a += 0.0f;                 // -0.0 and +0.0 move alike
    std::memcpy(&bv, &v, 4);
    std::memcpy(&ba, &a, 4);
    return ((uint64_t)bv << 32) | ba;
}

static int class_of(std::map<uint64_t, int32_t> &index, std::vector<AxisClass> &cls, float v, float a,
                    int32_t T, double t0, const float *times, const float *jitter, int axis, bool *ok) {
    const uint64_t key = key_of(v, a);
    auto it = index.find(key);
    if (it != index.end()) return it->second;
    AxisClass c;
    c.v = v; c.a = a;
    c.shift.resize(T);
    c.smin = INT32_MAX; c.smax = INT32_MIN;
    for (int32_t t = 0; t < T; ++t) {
        int32_t s = 0;
        const double dt = (times ? (double)times[t] : (double)t) - t0;
        const double j = jitter ? (double)jitter[2 * t + axis] : 0.0;
        bool tie = false;
        if (!axis_shift((double)v, (double)a, dt, j, &s, &tie)) { *ok = false; s = 0; }
        c.tie = c.tie || tie;
        c.jittered = c.jittered || j != 0.0;
        c.shift[t] = s;
        c.smin = std::min(c.smin, s);
        c.smax = std::max(c.smax, s);
    }
    const int32_t id = (int32_t)cls.size();
    cls.push_back(std::move(c));
    index.emplace(key, id);
    return id;
}

int build_classes(const tno_mf_traj *traj, int32_t n_traj, int32_t T, double t0, const float *frame_times,
                  const float *jitter_xy, Plan *plan) {
    plan->T = T;
    plan->t0 = t0;
    plan->xcls.clear(); plan->ycls.clear();
    plan->traj_xc.resize(n_traj);
    plan->traj_yc.resize(n_traj);
    std::map<uint64_t, int32_t> xi, yi;
    bool ok = true;
    for (int32_t k = 0; k < n_traj; ++k) {
        plan->traj_xc[k] = class_of(xi, plan->xcls, traj[k].vx, traj[k].ax, T, t0, frame_times, jitter_xy, 0, &ok);
        plan->traj_yc[k] = class_of(yi, plan->ycls, traj[k].vy, traj[k].ay, T, t0, frame_times, jitter_xy, 1, &ok);
    }
    return ok ? TNO_MF_OK : TNO_MF_EINVAL;
}

void build_batches(Plan *plan, int32_t max_entries, int32_t max_spread) {
    plan->batches.clear();
    const int32_t T = plan->T;
    const int32_t n_traj = (int32_t)plan->traj_xc.size();
    std::vector<std::vector<int32_t>> by_x(plan->xcls.size());
    for (int32_t k = 0; k < n_traj; ++k) by_x[plan->traj_xc[k]].push_back(k);
    std::vector<int32_t> lo(T), hi(T);
    for (size_t xc = 0; xc < by_x.size(); ++xc) {
        std::vector<int32_t> &ks = by_x[xc];
        std::stable_sort(ks.begin(), ks.end(), [&](int32_t p, int32_t q) {
            const AxisClass &cp = plan->ycls[plan->traj_yc[p]], &cq = plan->ycls[plan->traj_yc[q]];
            if (cp.v != cq.v) return cp.v < cq.v;
            return cp.a < cq.a;
        });
        Batch cur;
        cur.xcls = (int32_t)xc;
        cur.max_spread = 0;
        if (max_spread >= kUnlimitedSpread) {
            // no spread limit (the trajectory-following kernel): split the class into the fewest
            // batches, of sizes that differ by at most one
            const int32_t n = (int32_t)ks.size();
            const int32_t nbt = (n + max_entries - 1) / max_entries;
            int32_t pos = 0;
            for (int32_t j = 0; j < nbt; ++j) {
                const int32_t len = n / nbt + (j < n % nbt ? 1 : 0);
                cur.traj.assign(ks.begin() + pos, ks.begin() + pos + len);
                pos += len;
                for (int32_t t = 0; t < T; ++t) {
                    int32_t l = INT32_MAX, h = INT32_MIN;
                    for (int32_t k : cur.traj) {
                        const int32_t sh = plan->ycls[plan->traj_yc[k]].shift[t];
                        l = std::min(l, sh); h = std::max(h, sh);
                    }
                    cur.max_spread = std::max(cur.max_spread, h - l);
                }
                plan->batches.push_back(cur);
                cur.max_spread = 0;
            }
            continue;
        }
        for (int32_t k : ks) {
            const std::vector<int32_t> &s = plan->ycls[plan->traj_yc[k]].shift;
            bool fits = !cur.traj.empty() && (int32_t)cur.traj.size() < max_entries;
            int32_t spread = 0;
            if (fits) {
                for (int32_t t = 0; t < T; ++t) {
                    const int32_t l = std::min(lo[t], s[t]), h = std::max(hi[t], s[t]);
                    spread = std::max(spread, h - l);
                }
                fits = spread <= max_spread;
            }
            if (!fits) {
                if (!cur.traj.empty()) plan->batches.push_back(cur);
                cur.traj.clear();
                cur.max_spread = 0;
                for (int32_t t = 0; t < T; ++t) lo[t] = hi[t] = s[t];
            } else {
                for (int32_t t = 0; t < T; ++t) {
                    lo[t] = std::min(lo[t], s[t]);
                    hi[t] = std::max(hi[t], s[t]);
                }
                cur.max_spread = spread;
            }
            cur.traj.push_back(k);
        }
        if (!cur.traj.empty()) plan->batches.push_back(cur);
    }
}

void build_slot_batches(Plan *plan, int32_t max_slots, bool symmetric_filter) {
    plan->slot_batches.clear();
    const int32_t n_traj = (int32_t)plan->traj_xc.size();
    std::vector<std::vector<int32_t>> by_x(plan->xcls.size());
    for (int32_t k = 0; k < n_traj; ++k) by_x[plan->traj_xc[k]].push_back(k);
    struct Keyed { float v, a; int32_t pairable; Slot slot; };
    for (size_t xc = 0; xc < by_x.size(); ++xc) {
        std::vector<Keyed> slots;
        // orientation key (pairable, v, a) -> the slots that carry it, in order of creation
        std::map<std::pair<int32_t, uint64_t>, std::vector<size_t>> index;
        for (int32_t k : by_x[xc]) {
            const int32_t yc = plan->traj_yc[k];
            const AxisClass &c = plan->ycls[yc];
            const bool pairable = symmetric_filter && !c.tie && !c.jittered;
            float v = c.v + 0.0f, a = c.a + 0.0f;
            int32_t m = 0;
            if (pairable && (v < 0.0f || (v == 0.0f && a < 0.0f))) { v = -v; a = -a; m = 1; }
            std::vector<size_t> &list = index[std::make_pair((int32_t)pairable, key_of(v, a))];
            size_t found = SIZE_MAX;
            for (size_t i : list)
                if (slots[i].slot.member[m] < 0) { found = i; break; }
            if (found == SIZE_MAX) {
                Keyed ks;
                ks.v = v + 0.0f; ks.a = a + 0.0f; ks.pairable = pairable;
                ks.slot.member[0] = ks.slot.member[1] = -1;
                ks.slot.ycls = yc;
                ks.slot.flip = m;
                found = slots.size();
                slots.push_back(ks);
                list.push_back(found);
            }
            Slot &sl = slots[found].slot;
            sl.member[m] = k;
            // tables from the member in the slot's own orientation when there is one (the other one gives the
            // same numbers bit for bit: the class tables are odd in (v, a) when there is no tie)
            if (m == 0) { sl.ycls = yc; sl.flip = 0; }
        }
        std::stable_sort(slots.begin(), slots.end(), [](const Keyed &p, const Keyed &q) {
            if (p.v != q.v) return p.v < q.v;
            return p.a < q.a;
        });
        const int32_t n = (int32_t)slots.size();
        const int32_t nbt = (n + max_slots - 1) / max_slots;
        int32_t pos = 0;
        for (int32_t j = 0; j < nbt; ++j) {
            const int32_t len = n / nbt + (j < n % nbt ? 1 : 0);
            SlotBatch sb;
            sb.xcls = (int32_t)xc;
            for (int32_t i = 0; i < len; ++i) sb.slots.push_back(slots[pos + i].slot);
            pos += len;
            plan->slot_batches.push_back(std::move(sb));
        }
    }
}

}  // namespace tno
