// Host planner: axis classes and batches (see plan.h).  Compiled with -ffp-contract=off so that
// the displacement is evaluated exactly as on the device (separately rounded mul/add).
#include "plan.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <map>
#include <utility>

namespace tno {

bool axis_shift(double v, double a, double dt, double j, int32_t *shift) {
    volatile double p1 = v * dt;          // volatile: keep the operations separately rounded, in the
    volatile double adt = a * dt;         // order the device (tables.cu) and the oracle use
    volatile double p2 = adt * dt;
    volatile double d0 = p1 + p2;
    const double d = d0 + j;
    const double f = std::floor(d + 0.5);
    if (!(std::fabs(f) < 1.0e9)) return false;
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
        if (!axis_shift((double)v, (double)a, dt, j, &s)) { *ok = false; s = 0; }
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

}  // namespace tno
