// Host-side model of the tap-row ring protocol of the tensor-core engine (gm_tc.cuh): one MMA sequence that
// consumes, per window row y = Cfg::seq(i), the tap rows y - r (r = 0 .. kTileR-1), and one producer that
// issues tap rows in the order of the kernels' producer loop and may reuse a ring slot only after all kTileR
// uses of its previous tenant.  It uses the SAME constexpr mapping (seq, kNLow, slot_of) as the kernels and
// fails when the two sides wait for one another (the deadlock seen with 8-row tiles and rings split at NY / 2).
// Built and run by tests/test_tc_ring.py with nvcc (host code only; no GPU).
#include <cstdio>
#include <vector>

#include "gm_tc.cuh"

using namespace gm::tc;

template <int KP, int RING>
static int check(int jobs) {
  using C = Cfg<KP>;
  struct Tenant { int job, ta, left; };
  std::vector<Tenant> slot(2 * RING, Tenant{-1, -1, 0});
  std::vector<std::pair<int, int>> prod;                  // (job, tap row) in producer order
  for (int j = 0; j < jobs; ++j)
    for (int i = 0; i < C::NY; ++i) {
      const int y = C::seq(i);
      const int ta = (i & 1) ? y - (kTileR - 1) : y;
      if ((i & 1) ? (ta < C::kNLow || ta >= KP) : (ta >= C::kNLow)) continue;
      prod.push_back({j, ta});
    }
  if ((int)prod.size() != jobs * KP) { std::printf("KP=%d: producer loads %zu rows, not %d\n", KP, prod.size(), jobs * KP); return 1; }
  size_t pi = 0;
  for (int j = 0; j < jobs; ++j)
    for (int i = 0; i < C::NY;) {
      bool progressed = false;
      while (pi < prod.size()) {                            // the producer runs ahead as far as the ring lets it
        const int s = C::template slot_of<RING>(prod[pi].second);
        if (slot[s].left > 0) break;
        slot[s] = Tenant{prod[pi].first, prod[pi].second, kTileR};
        ++pi;
        progressed = true;
      }
      const int y = C::seq(i);
      bool ready = true;
      for (int r = 0; r < kTileR; ++r) {
        const int ta = y - r;
        if (ta < 0 || ta >= KP) continue;
        const Tenant& t = slot[C::template slot_of<RING>(ta)];
        if (t.job != j || t.ta != ta) ready = false;
      }
      if (ready) {
        for (int r = 0; r < kTileR; ++r) {
          const int ta = y - r;
          if (ta >= 0 && ta < KP) --slot[C::template slot_of<RING>(ta)].left;
        }
        ++i;
        progressed = true;
      }
      if (!progressed) { std::printf("DEADLOCK KP=%d RING=%d job %d step %d (window row %d)\n", KP, RING, j, i, y); return 1; }
    }
  for (const Tenant& t : slot)
    if (t.left != 0) { std::printf("KP=%d RING=%d: a tap row was used %d times too few\n", KP, RING, t.left); return 1; }
  return 0;
}

template <int KP>
static int check_all() {
  int bad = 0;
  bad += check<KP, kTileR + 1>(3);
  bad += check<KP, kTileR + 2>(3);
  bad += check<KP, 8>(3);
  bad += check<KP, kMaxRing>(3);
  bad += check<KP, Cfg<KP>::kRing>(3);
  return bad;
}

int main() {
  const int bad = check_all<9>() + check_all<17>() + check_all<25>() + check_all<33>() + check_all<41>();
  std::printf("tile %d x %d: %s\n", kTileR, kTileC, bad ? "FAILED" : "ok");
  return bad ? 1 : 0;
}
