// Host-only check of GqaPlan (csrc/attend_mma.cuh): the static + dynamic (or long + short, by SM class) ranges must partition the
// flattened list of cost units exactly, range_of() must invert range_lo() / range_hi(), and the walk a CTA makes
// over its range (gqa_piece, the function the kernel itself calls) must visit every (item, head, tile) exactly once,
// with the pieces of a pair numbered 0 .. last - first without a gap.  Built and run by tests/test_host_logic.py
// (nvcc, no GPU needed).
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "../../paper_2607_02640_b200/csrc/attend_mma.cuh"

using metronome::GqaPlan;
using metronome::GqaPiece;

// mode 0 static, 1 static + dynamic tail, 2 ranges by SM class (a random split of the CTAs into fast / slow, a random
// speed ratio): the launcher's own rules
static GqaPlan plan_for(int32_t Hkv, int64_t total, int64_t ctas, int mode, int32_t bnd) {
    if (mode < 2) return metronome::make_gqa_plan(Hkv, total, ctas, mode == 1, bnd);
    int64_t n_slow = 3 * (rand() % 60);
    if (n_slow >= ctas) n_slow = ctas - 1;
    const double ratio = 0.75 + 0.25 * (rand() % 1000) / 999.0;
    const GqaPlan g = metronome::make_gqa_plan_smclass(Hkv, total, ctas - n_slow, n_slow, ratio, bnd);
    if (g.n_total > ctas || g.n_static > ctas - n_slow) { printf("SM-class plan: %d ranges (%d long) for %lld CTAs (%lld fast)\n", g.n_total, g.n_static, (long long)ctas, (long long)(ctas - n_slow)); exit(1); }
    return g;
}

static int check(int64_t total, int64_t ctas, int mode, int32_t bnd) {
    const GqaPlan g = plan_for(4, total, ctas, mode, bnd);
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

// the kernel's walk, on the host: items with random tile counts, Hkv heads
static int walk(int n_items, int Hkv, int max_tiles, int64_t ctas, int mode, int32_t bnd) {
    const bool dynamic = mode == 1;
    std::vector<int32_t> n_tiles(n_items), tile_off(n_items);
    int64_t sum = 0;
    for (int i = 0; i < n_items; ++i) { n_tiles[i] = 1 + rand() % max_tiles; tile_off[i] = (int32_t)sum; sum += n_tiles[i]; }
    const int64_t total = (sum + (int64_t)bnd * n_items) * Hkv;
    if (ctas > sum * Hkv) ctas = sum * Hkv;
    const GqaPlan g = plan_for(Hkv, total, ctas, mode, bnd);
    std::vector<std::vector<int>> seen(n_items * Hkv);
    std::vector<std::vector<int>> pieces(n_items * Hkv);
    for (int i = 0; i < n_items; ++i) for (int h = 0; h < Hkv; ++h) seen[i * Hkv + h].assign(n_tiles[i], 0);
    for (int32_t r = 0; r < g.n_total; ++r) {
        int64_t u = g.range_lo(r);
        const int64_t u_end = g.range_hi(r);
        int32_t i = 0;                                                   // the host's range_item rule
        while (i + 1 < n_items && ((int64_t)tile_off[i + 1] + (int64_t)bnd * (i + 1)) * Hkv <= u) ++i;
        while (u < u_end) {
            if (i >= n_items) { printf("walked past the last item\n"); return 1; }
            const GqaPiece pc = metronome::gqa_piece(g, i, tile_off[i], n_tiles[i], u, u_end);
            if (pc.kvh < 0 || pc.kvh >= Hkv) { printf("head %d\n", pc.kvh); return 1; }
            if (pc.b <= pc.a) break;
            const int32_t first = g.range_of(pc.pair_lo), last = g.range_of(pc.pair_lo + n_tiles[i] - 1);
            if (r < first || r > last) { printf("range %d outside [%d, %d]\n", r, first, last); return 1; }
            if (last - first + 1 > g.max_pieces(n_tiles[i])) { printf("more pieces than max_pieces: n %d pieces %d max %d q1 %lld q2 %lld bnd %d dyn %d n_static %d n_total %d\n", n_tiles[i], last - first + 1, g.max_pieces(n_tiles[i]), (long long)g.q1, (long long)g.q2, bnd, (int)dynamic, g.n_static, g.n_total); return 1; }
            pieces[i * Hkv + pc.kvh].push_back(r - first);
            for (int t = pc.a; t < pc.b; ++t) ++seen[i * Hkv + pc.kvh][t];
            u = pc.pair_lo + pc.b;
            if (pc.kvh + 1 == Hkv) ++i;
        }
    }
    for (int i = 0; i < n_items; ++i)
        for (int h = 0; h < Hkv; ++h) {
            for (int t = 0; t < n_tiles[i]; ++t)
                if (seen[i * Hkv + h][t] != 1) { printf("item %d head %d tile %d visited %d times (bnd %d)\n", i, h, t, seen[i * Hkv + h][t], bnd); return 1; }
            const std::vector<int>& pp = pieces[i * Hkv + h];
            const int64_t pair_lo = ((int64_t)tile_off[i] + (int64_t)bnd * i) * Hkv + (int64_t)h * (n_tiles[i] + bnd) + bnd;
            const int want = g.range_of(pair_lo + n_tiles[i] - 1) - g.range_of(pair_lo) + 1;
            if ((int)pp.size() != want) { printf("item %d head %d: %d pieces, %d ranges\n", i, h, (int)pp.size(), want); return 1; }
            for (int k = 0; k < want; ++k) if (pp[k] != k) { printf("piece numbering\n"); return 1; }
        }
    return 0;
}

int main() {
    srand(260702640);
    int bad = 0, n = 0;
    for (int it = 0; it < 20000; ++it) {
        const int64_t ctas = 1 + rand() % 600;
        const int64_t total = ctas + rand() % 400000;
        const int32_t bnd = (it & 1) ? 8 : 0;
        bad += check(total, ctas, 0, bnd);
        if ((total + ctas - 1) / ctas >= 48) bad += check(total, ctas, 1, bnd);
        if (ctas >= 2) bad += check(total, ctas, 2, bnd);
        ++n;
    }
    bad += check(1, 1, 0, 0);
    bad += check(444, 444, 0, 8);
    bad += check(444, 444, 2, 8);
    const int32_t bnds[4] = {0, 1, 8, 16};
    for (int it = 0; it < 3000; ++it) {
        const int n_items = 1 + rand() % 200, Hkv = 1 + rand() % 8, max_tiles = (it % 3 == 0) ? 3 : 1 + rand() % 140;
        bad += walk(n_items, Hkv, max_tiles, 2 + rand() % 600, it % 3, bnds[it & 3]);
        ++n;
    }
    printf("%d cases, %d bad\n", n, bad);
    return bad ? 1 : 0;
}
