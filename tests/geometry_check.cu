// Host-only check of libge's tiling arithmetic (tests/test_geometry.py compiles and runs this on the CPU):
// for many shapes, every output node must be written by exactly one tile, every window must lie inside the
// rod, and the halo must cover the nodes that go stale in tb levels.  No kernel is launched.
#include <cstdio>
#include <cstdint>
#include <vector>

#include "../paper_1310_3422_b200/csrc/ge_temporal.cuh"
#include "../paper_1310_3422_b200/csrc/ge_strip2d.cuh"
#include "../paper_1310_3422_b200/csrc/ge_level_k.cuh"
#include "../paper_1310_3422_b200/csrc/ge_unit_k.cuh"

static int fails = 0;
#define CHECK(cond, ...) do { if (!(cond)) { if (fails < 20) { std::printf("FAIL %s: ", #cond); std::printf(__VA_ARGS__); std::printf("\n"); } ++fails; } } while (0)

// drift-free 1-D tiles (ge_temporal.cuh temporal1d_tile_df / ge_stream.cuh)
static void check_tiles_1d(int C, int V, int tb, int phase, int64_t nx) {
    const ge::Temporal1dGeom g = ge::temporal1d_geom(C, V, tb, phase);
    const int64_t W = 32 * (int64_t)C;
    if (nx < W || nx % V) return;
    const ge::Temporal1dTiles tl = ge::temporal1d_tiles(C, g, nx);
    const int stale = tb + g.pre + ((tb - g.pre) & 1);           // one per level, +1 for I, +1 for the shift back
    CHECK(g.halo >= stale && g.halo % V == 0 && g.valid % V == 0 && g.valid > 0 && g.valid + 2 * g.halo <= W,
          "C=%d tb=%d ph=%d halo=%d valid=%d", C, tb, phase, g.halo, g.valid);
    std::vector<int> hits((size_t)nx, 0);
    for (int64_t t = 0; t < tl.ntiles; ++t) {
        const bool first = t == 0, last = t == tl.nreg;
        const int64_t a0 = first ? 0 : (last ? nx - W : t * g.valid - g.halo);
        const int64_t lo = t * g.valid, hi = last ? nx : lo + g.valid;
        CHECK(a0 >= 0 && a0 + W <= nx && a0 % 2 == 0 && a0 % V == 0, "window C=%d tb=%d nx=%lld t=%lld a0=%lld", C, tb, (long long)nx, (long long)t, (long long)a0);
        // outputs must keep `stale` nodes away from a window edge that is not a boundary of the rod
        CHECK(first || lo - a0 >= stale, "left halo C=%d tb=%d nx=%lld t=%lld", C, tb, (long long)nx, (long long)t);
        CHECK(last || a0 + W - hi >= stale, "right halo C=%d tb=%d nx=%lld t=%lld", C, tb, (long long)nx, (long long)t);
        for (int64_t e = lo; e < hi; ++e) hits[(size_t)e]++;
    }
    for (int64_t e = 0; e < nx; ++e) if (hits[(size_t)e] != 1) { CHECK(false, "cover C=%d tb=%d ph=%d nx=%lld e=%lld hits=%d", C, tb, phase, (long long)nx, (long long)e, hits[(size_t)e]); break; }
}

// 2-D strips (ge_strip2d.cuh)
static void check_strips_2d(int C, int V, int TB, int64_t nx, int64_t ny, int hp) {
    if (nx < 32 * C || nx % 4) return;
    const ge::Strip2dGeom g = ge::strip2d_geom(C, V, TB, nx, ny, hp);
    CHECK(g.halo >= TB && g.valid > 0 && g.valid + 2 * g.halo <= 32 * C, "strip geom nx=%lld", (long long)nx);
    std::vector<int> hits((size_t)nx, 0);
    for (int s = 0; s < g.nstrips; ++s) {
        const bool first = s == 0, last = s == g.nreg;
        const int64_t a0 = first ? 0 : (last ? nx - 32 * C : (int64_t)s * g.valid - g.halo);
        const int64_t lo = (int64_t)s * g.valid, hi = last ? nx : lo + g.valid;
        CHECK(a0 >= 0 && a0 + 32 * C <= nx && a0 % V == 0, "strip window nx=%lld s=%d", (long long)nx, s);
        CHECK(first || lo - a0 >= TB, "strip left halo nx=%lld s=%d", (long long)nx, s);
        CHECK(last || a0 + 32 * C - hi >= TB, "strip right halo nx=%lld s=%d", (long long)nx, s);
        for (int64_t e = lo; e < hi; ++e) hits[(size_t)e]++;
    }
    for (int64_t e = 0; e < nx; ++e) if (hits[(size_t)e] != 1) { CHECK(false, "strip cover nx=%lld e=%lld hits=%d", (long long)nx, (long long)e, hits[(size_t)e]); break; }
    CHECK((int64_t)g.segs * 2 * hp >= ny && (int64_t)(g.segs - 1) * 2 * hp < ny, "segments ny=%lld hp=%d", (long long)ny, hp);
}

// units of the k >= 2 kernels (ge_level_k.cuh): every interior node belongs to exactly one unit
static void check_units(int k, int phase, int64_t nx) {
    const ge::LevelKGeom g = ge::level_k_geom(k, phase, nx, 8, 96 * 1024);
    if (g.upc < 1) return;
    std::vector<int> hits((size_t)nx + 2, 0);
    for (int64_t u = 0; u < g.units; ++u)
        for (int j = 0; j < 2 * k; ++j) { const int64_t i = g.s0 + u * 2 * k + j; if (i >= 1 && i <= nx) hits[(size_t)i]++; }
    for (int64_t i = 1; i <= nx; ++i) if (hits[(size_t)i] != 1) { CHECK(false, "units k=%d ph=%d nx=%lld i=%lld", k, phase, (long long)nx, (long long)i); break; }
    const ge::RodKGeom r = ge::rod_k_geom(k, nx, 8);
    CHECK(r.threads == 0 || r.threads >= g.units, "rod threads k=%d nx=%lld", k, (long long)nx);
}

// blocked k >= 2 kernels (r02): the shared-memory windows must deliver every node exactly once with at least
// tb (k+1) nodes between an output and a cut end of its window; the register form's tiles must deliver every unit
// exactly once with enough halo lanes, and the end windows must cover what the rod's ends spoil.
static void check_temporal_k(int k, int tb, int64_t nx) {
    const ge::TemporalKGeom g = ge::temporal_k_geom(k, tb, nx, 8, 64 * 1024);
    if (g.valid <= 0) return;
    CHECK(g.halo >= tb * (k + 1) && g.window == g.valid + 2 * g.halo && g.threads <= 1024 && g.threads * 2 * k >= g.window + 2 * k,
          "temporal_k geom k=%d tb=%d nx=%lld", k, tb, (long long)nx);
    CHECK(g.smem <= 64 * 1024 + 1024, "temporal_k smem k=%d tb=%d", k, tb);
    int64_t covered = 0;
    for (int64_t t = 0; t < g.tiles; ++t) {
        const int64_t v0 = 1 + t * g.valid, v1 = v0 + g.valid < nx + 1 ? v0 + g.valid : nx + 1;
        CHECK(v0 == covered + 1 && v1 > v0, "temporal_k cover k=%d nx=%lld t=%lld", k, (long long)nx, (long long)t);
        covered = v1 - 1;
    }
    CHECK(covered == nx, "temporal_k total k=%d tb=%d nx=%lld covered=%lld", k, tb, (long long)nx, (long long)covered);
}
static void check_unit_k(int k, int tb, int64_t nx) {
    const ge::UnitKGeom g = ge::unit_k_geom(k, tb, nx);
    if (g.valid_lanes < 64) return;
    CHECK(g.halo_lanes * 2 * k >= tb * (k + 1) + 2 * k, "unit halo k=%d tb=%d lanes=%d", k, tb, g.halo_lanes);
    const int64_t units = (nx + 2 * k - 1) / (2 * k);
    CHECK(g.tiles * g.valid_lanes >= units && (g.tiles - 1) * g.valid_lanes < units, "unit tiles k=%d nx=%lld", k, (long long)nx);
    // the end windows of ge_api.cu: tb (k+1) + 4k + 8 nodes, and their shared-memory window fits
    const int64_t end_len = (int64_t)tb * (k + 1) + 4 * k + 8;
    const ge::TemporalKGeom e = ge::temporal_k_ends_geom(k, tb, end_len, 8);
    CHECK(e.valid == end_len && e.threads * 2 * k >= e.window && e.smem <= 64 * 1024, "end windows k=%d tb=%d", k, tb);
    CHECK(end_len >= g.halo_lanes * 0 + tb * (k + 1) + 2 * k, "end length k=%d tb=%d", k, tb);
}
// cooperative 2-D strips: COOP warps share one strip
static void check_coop_strips(int C, int V, int TB, int COOP, int64_t nx) {
    if (nx < (int64_t)COOP * 32 * C || nx % 4) return;
    const ge::Strip2dGeom g = ge::strip2d_coop_geom(C, V, TB, COOP, nx, 64, 8);
    const int64_t W = (int64_t)COOP * 32 * C;
    std::vector<int> hits((size_t)nx, 0);
    for (int s = 0; s < g.nstrips; ++s) {
        const bool first = s == 0, last = s == g.nreg;
        const int64_t a0 = first ? 0 : (last ? nx - W : (int64_t)s * g.valid - g.halo);
        const int64_t lo = (int64_t)s * g.valid, hi = last ? nx : lo + g.valid;
        CHECK(a0 >= 0 && a0 + W <= nx && a0 % V == 0 && (first || lo - a0 >= TB) && (last || a0 + W - hi >= TB),
              "coop strip nx=%lld s=%d", (long long)nx, s);
        for (int64_t e = lo; e < hi; ++e) hits[(size_t)e]++;
    }
    for (int64_t e = 0; e < nx; ++e) if (hits[(size_t)e] != 1) { CHECK(false, "coop cover nx=%lld e=%lld hits=%d", (long long)nx, (long long)e, hits[(size_t)e]); break; }
}

int main() {
    for (int k : {2, 3, 5, 16, 64, 200}) for (int tb : {1, 4, 8, 16, 32}) for (int64_t nx : {40000, 70001, 262142, 1048576}) check_temporal_k(k, tb, nx);
    for (int k : {2, 4, 8, 16, 32}) for (int tb : {1, 5, 8, 16, 32, 48}) for (int64_t nx : {40000, 70001, 262142, 1048576, 268435456}) check_unit_k(k, tb, nx);
    for (int coop : {2, 4, 8}) for (int64_t nx : {512, 1024, 1032, 2600, 4104, 8192}) { check_coop_strips(4, 4, 6, coop, nx); check_coop_strips(2, 2, 6, coop, nx); }
    const int Cs64[] = {8, 16, 18, 22, 26, 32}, Cs32[] = {16, 32, 36, 44, 52, 64};
    const int64_t extra[] = {0, 2, 4, 8, 100, 576, 1000, 4098, 65536};
    for (int phase = 0; phase < 2; ++phase)
        for (int tb = 1; tb <= 64; tb += (tb < 24 ? 1 : 7)) {
            for (int C : Cs64) for (int64_t x : extra) { int64_t nx = 32 * C + x; nx -= nx % 2; if (tb <= ge::temporal1d_max_tb(C)) check_tiles_1d(C, 2, tb, phase, nx); }
            for (int C : Cs32) for (int64_t x : extra) { int64_t nx = 32 * C + x; nx -= nx % 4; if (tb <= ge::temporal1d_max_tb(C)) check_tiles_1d(C, 4, tb, phase, nx); }
        }
    for (int TB : {4, 6, 8}) for (int64_t nx : {128, 132, 232, 244, 256, 1000, 8192}) for (int64_t ny : {1, 7, 64, 1000}) for (int hp : {1, 5, 56, 64}) {
        check_strips_2d(4, 4, TB, nx, ny, hp);
        check_strips_2d(4, 2, TB, nx, ny, hp);
        check_strips_2d(2, 2, TB, nx, ny, hp);           // the fp64 default: 64-column strips
    }
    for (int TB : {4, 6, 8}) for (int64_t nx : {64, 68, 116, 120}) for (int64_t ny : {1, 7, 64}) for (int hp : {1, 5, 56})
        check_strips_2d(2, 2, TB, nx, ny, hp);
    for (int k : {2, 3, 5, 16, 64, 1000}) for (int phase = 0; phase < 2; ++phase) for (int64_t nx : {1, 2, 3, 30, 62, 8206, 100000}) check_units(k, phase, nx);
    // meetings of the whole-chip kernel: never more levels between two meetings than tb
    for (int tb = 2; tb <= 64; tb += 2) for (int64_t steps : {0, 1, 2, 3, 63, 64, 65, 1000, 10001}) for (int ph = 0; ph < 2; ++ph) {
        const int64_t m = ge::grid_resident_meetings(steps, ph, tb);
        CHECK(m >= (steps > tb + 2 ? (steps - 2) / tb - 1 : 0) && m <= steps / 2 + 1, "meetings steps=%lld tb=%d m=%lld", (long long)steps, tb, (long long)m);
    }
    // staggered meetings: a tile publishes every tbh levels and refreshes its halo every second publication,
    // so 2*tbh <= tb must hold; the host's count of publications (+ the final one) is the meeting loop at tbh
    for (int tb = 8; tb <= 128; tb += 2) for (int64_t steps : {0, 1, 2, 3, 63, 64, 65, 1000, 10001}) for (int ph = 0; ph < 2; ++ph) {
        const int tbh = tb / 2 - (tb / 2) % 2;
        CHECK(tbh >= 2 && 2 * tbh <= tb, "stagger tb=%d tbh=%d", tb, tbh);
        const int64_t h = ge::grid_resident_halves(steps, ph, tb);
        CHECK(h == ge::grid_resident_meetings(steps, ph, tbh) + 1, "halves steps=%lld tb=%d h=%lld", (long long)steps, tb, (long long)h);
    }
    std::printf("%s (%d failures)\n", fails ? "GEOMETRY FAILED" : "GEOMETRY OK", fails);
    return fails ? 1 : 0;
}
