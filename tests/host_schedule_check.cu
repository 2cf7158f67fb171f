// Host-side check of step a1 (the tile schedule): every decode used by the kernels is a bijection between the linear
// tile index and the block quadruples (full mode) / block-pair quadruples (split mode), in 32- and 64-bit arithmetic.
// Built and run by tests/test_schedule_host.py (no GPU needed: only __host__ code runs).
#include <cstdio>
#include <set>
#include <tuple>

#include "../paper_2310_04559_b200/csrc/ladder_ws.cuh"

using namespace ccl;

static int check_full(int nA, int nB, int nC, int nD, int SA, int SB, int SC, int SD, int idx32)
{
    FusedParams p = {};
    p.nA = nA; p.nB = nB; p.nC = nC; p.nD = nD;
    p.SA = SA; p.SB = SB; p.SC = SC; p.SD = SD;
    p.n_ab_blk = (long long)nA * nB; p.n_cd_blk = (long long)nC * nD; p.n_tiles = p.n_ab_blk * p.n_cd_blk;
    p.idx32 = idx32;
    std::set<std::tuple<int, int, int, int>> seen;
    for (long long T = 0; T < p.n_tiles; ++T) {
        int A, B, C, D;
        decode_tile4(p, T, A, B, C, D);
        if (A < 0 || A >= nA || B < 0 || B >= nB || C < 0 || C >= nC || D < 0 || D >= nD) return 1;
        if (!seen.insert(std::make_tuple(A, B, C, D)).second) return 2;
    }
    return (long long)seen.size() == p.n_tiles ? 0 : 3;
}

static int check_split(int nA, int nC, int H, int S, int idx32)
{
    FusedParams p = {};
    p.nA = p.nB = nA; p.nC = p.nD = nC;
    p.SA = p.SC = H; p.supertile = S;
    p.n_ab_blk = (long long)nA * (nA + 1) / 2; p.n_cd_blk = (long long)nC * (nC + 1) / 2;
    p.n_tiles = p.n_ab_blk * p.n_cd_blk;
    p.idx32 = idx32;
    std::set<std::tuple<int, int, int, int>> seen;
    for (long long T = 0; T < p.n_tiles; ++T) {
        long long ab, cd;
        decode_tile2(p, T, ab, cd);
        if (ab < 0 || ab >= p.n_ab_blk || cd < 0 || cd >= p.n_cd_blk) return 1;
        int A, B, C, D;
        decode_banded(ab, nA, H, A, B);
        decode_banded(cd, nC, H, C, D);
        if (A < 0 || A > B || B >= nA || C < 0 || C > D || D >= nC) return 2;
        if (!seen.insert(std::make_tuple(A, B, C, D)).second) return 3;
    }
    return (long long)seen.size() == p.n_tiles ? 0 : 4;
}

int main()
{
    int bad = 0;
    const int dims[][4] = {{1, 1, 1, 1}, {3, 2, 2, 3}, {5, 4, 3, 7}, {38, 25, 15, 38}, {7, 7, 7, 7}, {2, 9, 1, 4}};
    const int sts[][4] = {{3, 4, 3, 4}, {1, 1, 1, 1}, {2, 3, 2, 3}, {64, 64, 64, 64}, {1, 2, 1, 2}};
    for (auto &d : dims)
        for (auto &s : sts)
            for (int i32 = 0; i32 < 2; ++i32) {
                if (d[0] == 38 && i32 == 0 && s[0] != 3) continue;      // keep the run short
                const int rc = check_full(d[0], d[1], d[2], d[3], s[0], s[1], s[2], s[3], i32);
                if (rc) { printf("full %d %d %d %d / %d %d %d %d idx32=%d: rc %d\n", d[0], d[1], d[2], d[3], s[0], s[1], s[2], s[3], i32, rc); ++bad; }
            }
    for (int nA : {1, 2, 5, 19, 38})
        for (int nC : {1, 3, 10})
            for (int H : {1, 3, 4})
                for (int S : {1, 5, 12, 4096})
                    for (int i32 = 0; i32 < 2; ++i32) {
                        const int rc = check_split(nA, nC, H, S, i32);
                        if (rc) { printf("split nA %d nC %d H %d S %d idx32=%d: rc %d\n", nA, nC, H, S, i32, rc); ++bad; }
                    }
    // banded enumeration alone, and its locality: away from the diagonal H*W consecutive indices form an H x W rectangle
    for (int n = 1; n <= 40; ++n)
        for (int H = 1; H <= 5; ++H) {
            std::set<std::pair<int, int>> seen;
            const long long N = (long long)n * (n + 1) / 2;
            for (long long u = 0; u < N; ++u) {
                int r = -1, c = -1;
                decode_banded(u, n, H, r, c);
                if (r < 0 || c < r || c >= n || !seen.insert({r, c}).second) ++bad;
            }
        }
    {
        std::set<int> rows, cols;
        for (long long u = 30; u < 42; ++u) { int r, c; decode_banded(u, 20, 3, r, c); rows.insert(r); cols.insert(c); }
        if (rows.size() != 3 || cols.size() != 4) { printf("locality: %zu rows x %zu cols\n", rows.size(), cols.size()); ++bad; }
    }
    // packed-triangle layout of the split workspace (tri_base / tri_size): row c owns the slot d in [4*(c/4), v4); the
    // slots tile [0, tri_size) exactly once, every row base is a multiple of 4 (128-bit copies, full-sector reductions),
    // and the size is v^2/2 + O(v)
    for (int v : {1, 2, 3, 4, 5, 7, 8, 9, 20, 33, 37, 66, 120, 300, 420, 520}) {
        const long long v4 = tri_v4(v), nt = tri_size(v);
        std::set<long long> seen;
        for (int c = 0; c < v; ++c) {
            if (tri_base(c, v4) % 4) ++bad;
            for (long long d = (c & ~3); d < v4; ++d) {
                const long long k = tri_base(c, v4) + d;
                if (k < 0 || k >= nt || !seen.insert(k).second) ++bad;
            }
        }
        if ((long long)seen.size() != nt || nt % 4) { printf("tri layout v=%d: %zu slots of %lld\n", v, seen.size(), nt); ++bad; }
        if (v >= 66 && nt > (long long)(0.57 * v * v)) { printf("tri size v=%d: %lld\n", v, nt); ++bad; }
    }
    printf("bad=%d\n", bad);
    return bad ? 1 : 0;
}
