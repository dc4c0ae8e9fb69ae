// Host-side construction of the block-shell layout table of libnuma_b200.so (no CUDA).
#include <cmath>
#include <cstdint>
#include <utility>
#include <vector>

void numa_build_shell_pos(int N, int epb, int64_t BS, std::vector<int32_t> &pos,
                          std::vector<uint32_t> &tab);

// Block-shell position table (numa_internal.cuh, ShellLayout).  A block record holds the
// nodes of `epb` elements entity by entity (element interiors, the 6 face interiors, the 12
// edge interiors, the 8 corners; inside an entity element by element), padded to BS positions.
// The ORDER of the entities, the order of the nodes inside an entity and the place of the pad
// positions are free as far as the DSS is concerned (an entity stays one contiguous run), and
// are chosen so that the 16 nodes of every aligned 16-group of positions fall into 16 different
// 8-byte banks of the volume kernel's shared-memory work arrays (index sp = le*ME + i + SJ j +
// SK k): the pointwise phases of that kernel run one thread per POSITION, and a half-warp of
// 8-byte accesses is conflict-free exactly then.  Deterministic annealing (fixed LCG seed):
// the same table on every machine, hence bitwise reproducible DSS order.
#ifndef NUMA_SHELL_MAXRUN
#define NUMA_SHELL_MAXRUN 16
#endif
static const int kMaxRun = NUMA_SHELL_MAXRUN;
#ifndef NUMA_SHELL_ITERS
#define NUMA_SHELL_ITERS 2
#endif

void numa_build_shell_pos(int N, int epb, int64_t BS, std::vector<int32_t> &pos,
                          std::vector<uint32_t> &tab)
{
    const int Nq = N + 1, N2 = Nq * Nq, Mn = N2 * Nq;
    const int SJ = Nq, SK = (Nq & 1) ? N2 : N2 + 1, ME = SK * Nq;
    const int npb = epb * Mn, nb = (int)BS;
    std::vector<int> ent(Mn);
    for (int n = 0; n < Mn; ++n) {
        const int i = n % Nq, j = (n / Nq) % Nq, k = n / N2;
        const bool bi = (i == 0 || i == N), bj = (j == 0 || j == N), bk = (k == 0 || k == N);
        const int nbnd = bi + bj + bk;
        int id;
        if (nbnd == 0) id = 0;
        else if (nbnd == 1) id = 1 + (bi ? (i == N) : bj ? 2 + (j == N) : 4 + (k == N));
        else if (nbnd == 2) {
            const int free_dir = !bi ? 0 : !bj ? 1 : 2;
            const int sd = (free_dir == 0) ? (j == N) + 2 * (k == N)
                         : (free_dir == 1) ? (i == N) + 2 * (k == N) : (i == N) + 2 * (j == N);
            id = 7 + 4 * free_dir + sd;
        } else id = 19 + (i == N) + 2 * (j == N) + 4 * (k == N);
        ent[n] = id;
    }
    auto bank_of = [&](int bn) {   // bn = le*Mn + n
        const int le = bn / Mn, n = bn % Mn;
        const int i = n % Nq, j = (n / Nq) % Nq, k = n / N2;
        return (le * ME + i + SJ * j + SK * k) & 15;
    };
    // movable blocks: the 26 boundary entities, every interior node, every pad position
    std::vector<std::vector<int>> blocks;
    for (int e = 0; e < 27; ++e) {
        std::vector<int> b;
        for (int le = 0; le < epb; ++le)
            for (int n = 0; n < Mn; ++n)
                if (ent[n] == e) b.push_back(le * Mn + n);
        if (b.empty()) continue;
        // element-interior nodes are shared with nobody: the DSS never touches them, so they need
        // not stay together and serve as free filler between the face / edge / corner runs
        if (e == 0) { for (int x : b) blocks.push_back(std::vector<int>(1, x)); continue; }
        // a face interior longer than kMaxRun is cut into equal runs (still >= 12 nodes = three
        // sectors each): inside one long face run too few banks occur for a conflict-free warp
        const int parts = ((int)b.size() + kMaxRun - 1) / kMaxRun;
        for (int q = 0; q < parts; ++q) {
            const size_t lo = b.size() * q / parts, hi = b.size() * (q + 1) / parts;
            blocks.push_back(std::vector<int>(b.begin() + lo, b.begin() + hi));
        }
    }
    for (int t = npb; t < nb; ++t) blocks.push_back(std::vector<int>(1, -1));
#ifndef NUMA_SHELL_COMPACT_MINN
#define NUMA_SHELL_COMPACT_MINN 4
#endif
    // COMPACT (N >= 4): all face / edge / corner runs at the front of the record -- one contiguous
    // region per element and field that the DSS touches, so its 32-byte sectors and DRAM bursts are
    // fully used -- interior nodes and pads behind them; blocks then only trade places inside their
    // zone.  The price is bank conflicts in the volume kernel's pointwise phases (wavefront ratio
    // 1.25 / 1.5 / 1.6 / 1.8 / 1.2 at N = 4..8 instead of 1.0-1.3), which cost it 0-2 %; measured per
    // 32 M nodes (DSS ms, stage fraction): N=4 0.54 -> 0.52 (0.68 -> 0.69), N=5 0.60 -> 0.52 (0.64 -> 0.66),
    // N=7 0.50 -> 0.39 (0.61 -> 0.64), N=8 0.47 -> 0.37 (0.57 -> 0.60); N=3 neutral (left interleaved).
    std::vector<int> zone(blocks.size(), 0);
    if (N >= NUMA_SHELL_COMPACT_MINN) {
        std::vector<std::vector<int>> sh, in;
        for (auto &b : blocks) ((b.size() > 1 || (b[0] >= 0 && ent[b[0] % Mn] != 0)) ? sh : in).push_back(b);
        blocks = sh;
        blocks.insert(blocks.end(), in.begin(), in.end());
        for (size_t b = 0; b < blocks.size(); ++b) zone[b] = b < sh.size() ? 1 : 0;
    }
    std::vector<int> seq(nb), start(blocks.size());
    auto flatten = [&]() {
        int t = 0;
        for (size_t b = 0; b < blocks.size(); ++b) {
            start[b] = t;
            for (int x : blocks[b]) seq[t++] = x;
        }
    };
    constexpr int GW = 32;   // a warp: its two half-warps may take any 16 + 16 split of the group
    const int ng = (nb + GW - 1) / GW;
    std::vector<int> gc(ng);
    auto group_cost = [&](int g) {   // nodes that a bank holds beyond two
        int cnt[16] = {0}, c = 0;
        for (int t = GW * g; t < GW * g + GW && t < nb; ++t) {
            if (seq[t] < 0) continue;
            if (++cnt[bank_of(seq[t])] > 2) ++c;
        }
        return c;
    };
    // the quantity that matters: wavefronts of a thread-per-position 8-byte access, i.e. per
    // half-warp the largest number of nodes in one bank, after the lanes have been dealt as below
    auto wavefronts_ideal = [&]() {
        for (int g = 0; g < ng; ++g)
            if (group_cost(g) > 0) return false;
        return true;
    };
    uint64_t rng = 0x9E3779B97F4A7C15ull;
    auto rnd = [&]() { rng = rng * 6364136223846793005ull + 1442695040888963407ull; return (uint32_t)(rng >> 33); };
    flatten();
    int cur = 0;
    for (int g = 0; g < ng; ++g) cur += (gc[g] = group_cost(g));
    const int nblk = (int)blocks.size();
    // measured (pointwise wavefronts over the ideal two per request): 1.00 at N <= 5, 1.0-1.05 at
    // N = 6 and 8; N = 7 (no pad positions, 16 nodes of every 8-byte bank pair) stays near 1.2
    // (N = 8: three times longer -- its 736-thread block is alone on the SM and feels the conflicts:
    //  wavefront ratio 1.30 -> 1.13, stage fraction 0.597 -> 0.605)
    const long iters = (nb > 128 ? NUMA_SHELL_ITERS * (N == 8 ? 3 : 1) : 1) * (400000L + 4000L * nb);
    auto accept_step = [&](int delta, long it) {
        if (delta <= 0) return true;
        // accept an uphill step of d with probability 2^(-d / T), T falling linearly
        const double T = 0.8 * (1.0 - (double)it / iters) + 0.05;
        const double pr = std::exp2(-(double)delta / T);
        return (rnd() & 0xffff) < (uint32_t)(pr * 65536.0);
    };
    for (long it = 0; it < iters && cur > 0; ++it) {
        if ((it & 65535) == 0 && wavefronts_ideal()) break;
        const uint32_t mv = rnd() & 31;
        if (mv < 8) {
            // swap two whole blocks (mostly two of equal length: cheap); a general swap moves
            // every group between them
            int a = (int)(rnd() % nblk), b = (int)(rnd() % nblk);
            if (mv >= 4) {
                for (int tries = 0; tries < 4 && blocks[a].size() != blocks[b].size(); ++tries) b = (int)(rnd() % nblk);
                if (blocks[a].size() != blocks[b].size()) continue;
            }
            if (a == b || zone[a] != zone[b]) continue;
            if (a > b) std::swap(a, b);
            if (blocks[a].size() == blocks[b].size()) {
                // equal lengths: the other blocks stay where they are, only the groups under the
                // two blocks change
                const int L = (int)blocks[a].size();
                int gs[8], ng2 = 0;
                auto add_groups = [&](int s0) {
                    for (int g = s0 / GW; g <= (s0 + L - 1) / GW; ++g) {
                        bool seen = false;
                        for (int q = 0; q < ng2; ++q) seen |= (gs[q] == g);
                        if (!seen && ng2 < 8) gs[ng2++] = g;
                    }
                };
                add_groups(start[a]); add_groups(start[b]);
                int old = 0;
                for (int q = 0; q < ng2; ++q) old += gc[gs[q]];
                for (int t = 0; t < L; ++t) std::swap(seq[start[a] + t], seq[start[b] + t]);
                int nw = 0, cs[8];
                for (int q = 0; q < ng2; ++q) nw += (cs[q] = group_cost(gs[q]));
                if (accept_step(nw - old, it)) {
                    std::swap(blocks[a], blocks[b]);
                    for (int q = 0; q < ng2; ++q) gc[gs[q]] = cs[q];
                    cur += nw - old;
                } else {
                    for (int t = 0; t < L; ++t) std::swap(seq[start[a] + t], seq[start[b] + t]);
                }
                continue;
            }
            const int lo = start[a] / GW;
            const int hi = (start[b] + (int)blocks[b].size() - 1) / GW;
            int old = 0;
            for (int g = lo; g <= hi; ++g) old += gc[g];
            std::swap(blocks[a], blocks[b]);
            flatten();
            int nw = 0;
            for (int g = lo; g <= hi; ++g) nw += group_cost(g);
            if (accept_step(nw - old, it)) {
                for (int g = lo; g <= hi; ++g) gc[g] = group_cost(g);
                cur += nw - old;
            } else {
                std::swap(blocks[a], blocks[b]);
                flatten();
            }
        } else {
            // swap two nodes inside one block: at most two groups change
            const int bi = (int)(rnd() % nblk);
            const int L = (int)blocks[bi].size();
            if (L < 2) continue;
            const int a = (int)(rnd() % L), b = (int)(rnd() % L);
            if (a == b) continue;
            const int pa = start[bi] + a, pb = start[bi] + b, ga = pa / GW, gb = pb / GW;
            if (ga == gb) continue;   // same group: the cost cannot change
            const int old = gc[ga] + gc[gb];
            std::swap(seq[pa], seq[pb]);
            const int ca = group_cost(ga), cb = group_cost(gb);
            if (accept_step(ca + cb - old, it)) {
                std::swap(blocks[bi][a], blocks[bi][b]);
                gc[ga] = ca; gc[gb] = cb;
                cur += ca + cb - old;
            } else {
                std::swap(seq[pa], seq[pb]);
            }
        }
    }
    flatten();
    // thread slot -> position: inside every warp's 32 positions the lanes are dealt so that
    // each half-warp (lanes 0-15, 16-31) gets at most one node of a bank where the group allows
    pos.assign((size_t)npb, 0);
    tab.assign((size_t)nb, 0xFFFFFFFFu);
    for (int g = 0; g < ng; ++g) {
        int half_of[GW], nh[2] = {0, 0};
        for (int l = 0; l < GW; ++l) half_of[l] = -1;
        // bank by bank (fullest first), the nodes of a bank alternate between the two halves,
        // starting with the emptier half: two nodes of a bank never meet unless it holds > 2
        std::vector<int> by_bank[16];
        for (int l = 0; l < GW && GW * g + l < nb; ++l)
            if (seq[GW * g + l] >= 0) by_bank[bank_of(seq[GW * g + l])].push_back(l);
        int order16[16];
        for (int b2 = 0; b2 < 16; ++b2) order16[b2] = b2;
        for (int x = 0; x < 16; ++x)          // selection sort, descending size, stable
            for (int y = x + 1; y < 16; ++y)
                if (by_bank[order16[y]].size() > by_bank[order16[x]].size()) std::swap(order16[x], order16[y]);
        for (int x = 0; x < 16; ++x) {
            const std::vector<int> &v = by_bank[order16[x]];
            const int h0 = (nh[0] <= nh[1]) ? 0 : 1;
            for (size_t r2 = 0; r2 < v.size(); ++r2) {
                int h = h0 ^ (int)(r2 & 1);
                if (nh[h] >= GW / 2) h ^= 1;
                half_of[v[r2]] = h;
                nh[h]++;
            }
        }
        int next[2] = {0, GW / 2};
        for (int l = 0; l < GW && GW * g + l < nb; ++l) {
            const int t = GW * g + l, bn = seq[t];
            if (bn < 0) continue;                            // pad position: no thread works on it
            int h = half_of[l];
            if (next[h] >= (h ? GW : GW / 2)) h ^= 1;
            const int slot = GW * g + next[h]++;
            pos[(size_t)bn] = t;
            const int le = bn / Mn, n = bn % Mn;
            const int i = n % Nq, j = (n / Nq) % Nq, k = n / N2;
            tab[(size_t)slot] = (uint32_t)(le * ME + i + SJ * j + SK * k) | ((uint32_t)i << 10) |
                                ((uint32_t)j << 14) | ((uint32_t)k << 18) | ((uint32_t)le << 22) |
                                ((uint32_t)l << 26);
        }
    }
}
