// Host-only check of GqaPlan (csrc/attend_mma.cuh): the static + dynamic ranges must partition the
// flattened tile list exactly, and range_of() must invert range_lo() / range_hi().  Built and run by
// tests/test_host_logic.py (nvcc, no GPU needed).
#include <cstdio>
#include <cstdlib>
#include "../../paper_2607_02640_b200/csrc/attend_mma.cuh"

using metronome::GqaPlan;

static int check(int64_t total, int64_t ctas, bool dynamic) {
    const GqaPlan g = metronome::make_gqa_plan(4, total, ctas, dynamic);      // the launcher's own rule
    int64_t expect = 0;
    for (int32_t r = 0; r < g.n_total; ++r) {
        const int64_t lo = g.range_lo(r), hi = g.range_hi(r);
        if (lo != expect || hi < lo || hi > total) { printf("range %d [%lld, %lld) expected lo %lld\n", r, (long long)lo, (long long)hi, (long long)expect); return 1; }
        if (hi > lo && (g.range_of(lo) != r || g.range_of(hi - 1) != r)) { printf("range_of mismatch at range %d\n", r); return 1; }
        expect = hi;
    }
    if (expect != total) { printf("covered %lld of %lld\n", (long long)expect, (long long)total); return 1; }
    if (g.max_pieces(1) < 1) return 1;
    return 0;
}

int main() {
    srand(260702640);
    int bad = 0, n = 0;
    for (int it = 0; it < 20000; ++it) {
        const int64_t ctas = 1 + rand() % 600;
        const int64_t total = ctas + rand() % 400000;
        bad += check(total, ctas, false);
        if ((total + ctas - 1) / ctas >= 48) bad += check(total, ctas, true);
        ++n;
    }
    bad += check(1, 1, false);
    bad += check(444, 444, false);
    printf("%d cases, %d bad\n", n, bad);
    return bad ? 1 : 0;
}
