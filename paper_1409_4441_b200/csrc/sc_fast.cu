// sc_fast.cu -- host side of the fast kernels: ring-pair tables (the ring-range disc query: input rings and azimuthal
// half windows of every base ring), tile lists of the sym kernel (sc_sym.cuh) and of the belt kernel (sc_belt.cu),
// kernel variant selection, launches over the whole sphere, latitude chunks (pipelined host entry) and latitude bands.
#include "sc_fast.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <vector>

namespace sc {

constexpr int kSymChunksDflt = 5;  // latitude chunks of the cap rings for the pipelined host entry
constexpr int kBeltChunksDflt = 6; // same for the belt rings
constexpr int kSymBufH = 2;        // stage buffers of the sym kernel (kSymBuf in sc_sym.cuh)

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
size_t belt_smem_bytes(int NC, int slack, int px, int nbuf, int ntb, int pw_max, int ne_max);
cudaError_t launch_belt(const Dev &P, const BeltDev &F, const Maps &io, int B, int threads, int slack, int px, size_t smem, int nsm,
                        cudaStream_t st);

// Host geometry kept for building tile lists after plan creation (latitude bands)
struct HostGeo {
    int N = 0, polar = 0;
    std::vector<std::vector<PairEnt>> per_ring;   // per base ring 1 .. 2N: its input rings
    std::vector<int> slot_of, pair_off;           // base ring -> slot; slot -> first entry of `pairs`
    std::vector<char> is_belt;
    int ipof(int r) const { return r < N ? r : (r <= 3 * N ? N : 4 * N - r); }
    int shof(int r) const { return (r >= N && r <= 3 * N) ? ((r - N) & 1) : 0; }
};

// Sym-kernel tiles of the non-belt base rings r_lo .. r_hi, longest first, appended to `tiles`.  Tiles are
// packed from runs of base pixels on one ring (32 R pixels per warp): whole runs of `run` pixels first, the
// ragged remainders are bin-packed (first fit, decreasing); a tile holds at most W warps, kMaxSub runs and
// Llimit staged positions (shared memory).  Returns the staged positions the tiles need.
// mirror: base pixels are the first half of the quadrant only, k = 0 .. (ip - 1 + sh) / 2 (the other half are their
// reflections phi -> pi/2 - phi, computed by the same threads).
// all_rings: also the base rings that the belt kernel normally takes (north-cap-only convolution).
// lanes: lanes of a warp that own a group of R base pixels each (32; 16 in the lane-pair instance).
static int build_sym_tiles(const HostGeo &g, int R, int W, int run, int Llimit, int r_hi, int r_lo, bool mirror,
                           std::vector<SymTile> &tiles, bool all_rings = false, int lanes = 32, int wcap = 0, int pad = 0, bool skew = false) {
    const int C = lanes * R;
    struct SubH { int r, k0, n, nw; int Lcap; double work; };
    auto make_sub = [&](int r, int k0, int n) {
        SubH sb{r, k0, n, (n + C - 1) / C, 0, 0.0};
        const int ip = g.ipof(r), sh = g.shof(r);
        const int klast = k0 + n - 1;
        for (const PairEnt &pe : g.per_ring[r]) {
            const int w0 = ((2 * k0 + 1 - sh) * pe.ipq + pe.shq * ip) / (2 * ip) - pe.hw;
            const int L = ((2 * klast + 1 - sh) * pe.ipq + pe.shq * ip) / (2 * ip) + pe.hw + R - w0 + (skew ? 2 * pe.ex : 0);      // skew: runs staged ex positions further on both sides
            sb.Lcap = std::max(sb.Lcap, L);
            sb.work += (double)(2 * pe.hw + R);
        }
        sb.Lcap = ((sb.Lcap + 7) & ~7) + pad;           // pad: alignment slack of the planar instances' bulk copies
        sb.work *= sb.nw;
        return sb;
    };
    std::vector<std::vector<SubH>> bins;
    std::vector<SubH> partial;
    for (int r = r_hi; r >= r_lo; --r) {
        if (r <= g.polar || (g.is_belt[r] && !all_rings)) continue;
        const int ip = mirror ? (g.ipof(r) + 1 + g.shof(r)) / 2 : g.ipof(r);     // base pixels of this ring
        int k0 = 0;
        for (; ip - k0 >= run; k0 += run) bins.push_back({make_sub(r, k0, run)});
        if (k0 < ip) partial.push_back(make_sub(r, k0, ip - k0));
    }
    const size_t nfull = bins.size();
    std::stable_sort(partial.begin(), partial.end(), [](const SubH &a, const SubH &b) { return a.nw > b.nw; });
    const int Wcap = wcap > 0 ? std::min(W, wcap) : W;   // warps per packed tile (< W only for small maps: runs shortened to spread over the SMs)
    std::vector<int> used(nfull, W), lsum(nfull, 0);
    for (const SubH &sb : partial) {
        size_t i = nfull;
        for (; i < bins.size(); ++i)
            if (used[i] + sb.nw <= Wcap && (int)bins[i].size() < kMaxSub && lsum[i] + sb.Lcap <= Llimit) break;
        if (i == bins.size()) { bins.emplace_back(); used.push_back(0); lsum.push_back(0); }
        bins[i].push_back(sb); used[i] += sb.nw; lsum[i] += sb.Lcap;
    }
    std::vector<std::pair<double, size_t>> order;
    int Lneed = 0;
    for (size_t i = 0; i < bins.size(); ++i) {
        double w = 0; int L = 0;
        for (const SubH &sb : bins[i]) { w = std::max(w, sb.work / sb.nw); L += sb.Lcap; }
        order.push_back({-w, i});
        Lneed = std::max(Lneed, L);
    }
    std::stable_sort(order.begin(), order.end());
    const size_t t0 = tiles.size();
    tiles.resize(t0 + bins.size());
    for (size_t t = 0; t < order.size(); ++t) {
        const std::vector<SubH> &bn = bins[order[t].second];
        SymTile &tl = tiles[t0 + t];
        std::memset(&tl, 0, sizeof(tl));
        tl.nsub = (int)bn.size();
        int w0 = 0, soff = 0;
        for (int i = 0; i < tl.nsub; ++i) {
            const SubH &sb = bn[i];
            const int slot = g.slot_of[sb.r];
            tl.sub[i] = SubTile{sb.r, sb.k0, sb.n, g.pair_off[slot], g.pair_off[slot + 1] - g.pair_off[slot], w0, sb.nw, soff};
            tl.nsteps = std::max(tl.nsteps, tl.sub[i].ne);
            w0 += sb.nw; soff += sb.Lcap;
        }
        tl.pad0 = soff;                                  // staged slots of the tile
    }
    return Lneed;
}

struct FastCfg {            // per batch size
    bool ok = false;
    int threads = 0, R = 1, Ltot = 0;
    size_t smem = 0;
    SymTile *tiles = nullptr;     // [0, ntiles): all rings, work sorted; then the latitude chunks
    int ntiles = 0, ntiles_all = 0, run = 0;
    bool tmem = false;            // 384-consumer variant with the running totals in tensor memory (large discs)
    bool tot = true;              // second accumulator set (per-ring partial sums added to running totals)
    bool mirror = false;          // 16 images per pair geometry (reflection phi -> pi/2 - phi as well)
    bool pair = false;            // lane-pair instance: 16 lane pairs x R base pixels per warp
    bool planar = false;          // planar staging by TMA bulk copies (sc_sym_pl.cu)
    bool skew = false;            // lane skew (planar and batch instances): longer staged runs
    std::map<std::pair<int, int>, std::pair<SymTile *, int>> band_tiles;   // (ring lo, hi) -> device tile list
    std::vector<int> ch_off, ch_lo, ch_hi;   // chunk i: tiles [ch_off[i], ch_off[i+1]), base rings ch_lo[i] .. ch_hi[i]
};

struct FastPlan {
    PairEnt *pairs = nullptr;
    int ntab_s = 0;
    int polar = 0;
    int first_belt = 0;           // base rings first_belt .. 2N go to the belt kernel (2N + 1: none)
    FastCfg cfg[kMaxB + 1];
    std::map<int, FastCfg> caps;  // north-only instances (sc_convolve_cap) by last ring, one map per launch; built on first use
    size_t tab_bytes = 0;
    int smem_optin = 0;
    double mean_nb = 0.0;         // mean number of pixels per disc
    int nsm = 148;
    // belt kernel
    bool belt_ok = false;
    BeltDev belt{};
    int belt_threads = 0;
    size_t belt_smem = 0;
    int *pair_off = nullptr;
    int *woff = nullptr;
    int4 *belt_tiles = nullptr;
    std::vector<int> bch_off, bch_lo, bch_hi;   // belt latitude chunks (tile offsets, base rings), equator first
    std::shared_ptr<HostGeo> geo;
    int belt_tiles_per_ring = 0, belt_slack = 0, belt_px = 4;   // belt_px: pixels per consumer thread (4 x 8 images or 8 x 4)
    int *grp_off = nullptr, *grp_e = nullptr;
    int *tile_ctr = nullptr;      // device counter of the sym kernel's dynamic tile schedule
    PairEntD *pairsd = nullptr;   // fp64 ring pairs (Dev::hp plans)
};

// the sym kernel instance of this batch size over a tile list
static cudaError_t dispatch_sym(const FastPlan *fp, const FastCfg &c, const Dev &P, const Maps &io, int B, cudaStream_t st,
                                const SymTile *tiles, int nt, bool south = true, bool overlap = false) {
    if (nt <= 0) return cudaSuccess;
    const SymLaunch L{fp->pairs, tiles, nt, c.Ltot, fp->ntab_s, fp->nsm, c.threads, c.R, c.smem, c.tot, c.tmem, c.mirror, south, c.pair, fp->tile_ctr, fp->pairsd, overlap, c.planar};
    if (c.planar) return B == 1 ? dispatch_sym_pl(L, P, io, st) : cudaErrorInvalidValue;
    if (c.pair) return B == 1 ? dispatch_sym_pair(L, P, io, st) : cudaErrorInvalidValue;
    return B == 1 ? dispatch_sym_b1(L, P, io, st) : dispatch_sym_bn(L, P, io, B, st);
}

// which: bit 0 = sym kernel, bit 1 = belt kernel (the two write disjoint pixels and may run on different
// streams); chunk < 0: all tiles (work sorted), else latitude chunk `chunk` of that kernel
cudaError_t fast_launch(FastPlan *fp, const Dev &P, const Maps &io, int B, int which, cudaStream_t st, int *launches,
                        int chunk) {
    *launches = 0;
    if (!fp || B < 1 || B > kMaxB || !fp->cfg[B].ok) return cudaErrorInvalidValue;
    const FastCfg &c = fp->cfg[B];
    cudaError_t e = cudaSuccess;
    if (which & 1) {
        int t0 = 0, nt = c.ntiles;
        if (chunk >= 0) {
            if (chunk + 1 >= (int)c.ch_off.size()) return cudaErrorInvalidValue;
            t0 = c.ch_off[chunk]; nt = c.ch_off[chunk + 1] - t0;
        }
        if ((e = dispatch_sym(fp, c, P, io, B, st, c.tiles + t0, nt)) != cudaSuccess) return e;
        *launches += nt > 0 ? 1 : 0;
    }
    if ((which & 2) && fp->belt_ok) {
        BeltDev F = fp->belt;
        if (chunk >= 0) {
            if (chunk + 1 >= (int)fp->bch_off.size()) return cudaErrorInvalidValue;
            F.tiles += fp->bch_off[chunk]; F.ntiles = fp->bch_off[chunk + 1] - fp->bch_off[chunk];
        }
        if (F.ntiles > 0) {
            e = launch_belt(P, F, io, B, fp->belt_threads, fp->belt_slack, fp->belt_px, fp->belt_smem, fp->nsm, st);
            if (e == cudaSuccess) ++*launches;
        }
    }
    return e;
}

// Latitude band: the fast kernels over base rings lo .. hi only (1 <= lo <= hi <= 2N; their southern mirrors
// included).  The sym tile list of a band is built on first use and cached (synchronous the first time).
cudaError_t fast_launch_band(FastPlan *fp, const Dev &P, const Maps &io, int B, int lo, int hi, cudaStream_t st,
                             int *launches) {
    *launches = 0;
    if (!fp || B < 1 || B > kMaxB || !fp->cfg[B].ok) return cudaErrorInvalidValue;
    FastCfg &c = fp->cfg[B];
    const int N = P.nside;
    cudaError_t e = cudaSuccess;
    const int s_lo = std::max(lo, fp->polar + 1), s_hi = std::min(hi, std::min(fp->first_belt - 1, 2 * N));
    if (s_lo <= s_hi) {
        auto it = c.band_tiles.find({s_lo, s_hi});
        if (it == c.band_tiles.end()) {
            std::vector<SymTile> tiles;
            const int Lneed = build_sym_tiles(*fp->geo, c.R, c.threads / 32, c.run, c.Ltot, s_hi, s_lo, c.mirror, tiles, false, c.pair ? 16 : 32, 0, c.planar ? kPlanarPad : 0, c.skew);
            if (Lneed > c.Ltot) return cudaErrorInvalidValue;
            SymTile *d = nullptr;
            if ((e = cudaMalloc((void **)&d, std::max<size_t>(tiles.size(), 1) * sizeof(SymTile))) != cudaSuccess) return e;
            if (!tiles.empty() && (e = cudaMemcpy(d, tiles.data(), tiles.size() * sizeof(SymTile), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
            it = c.band_tiles.emplace(std::make_pair(s_lo, s_hi), std::make_pair(d, (int)tiles.size())).first;
        }
        if (it->second.second > 0) {
            if ((e = dispatch_sym(fp, c, P, io, B, st, it->second.first, it->second.second)) != cudaSuccess) return e;
            ++*launches;
        }
    }
    const int b_lo = std::max(lo, fp->first_belt), b_hi = std::min(hi, 2 * N);
    if (fp->belt_ok && b_lo <= b_hi) {
        BeltDev F = fp->belt;                               // tile list: ring 2N first, belt_tiles_per_ring tiles per ring
        F.tiles += (2 * N - b_hi) * fp->belt_tiles_per_ring;
        F.ntiles = (b_hi - b_lo + 1) * fp->belt_tiles_per_ring;
        e = launch_belt(P, F, io, B, fp->belt_threads, fp->belt_slack, fp->belt_px, fp->belt_smem, fp->nsm, st);
        if (e == cudaSuccess) ++*launches;
    }
    return e;
}

// North cap only (a partial-sky map oriented so that the survey area lies in the polar cap): base rings
// polar + 1 .. ring_hi of the NORTHERN hemisphere, one map, through the north-only instance of the sym kernel (4 rotations
// x mirror = 8 images per pair geometry; nothing south of the disc of ring ring_hi is read).  The instance shape and the
// tile list of a given ring_hi are built on first use and cached (synchronous the first time).
cudaError_t fast_launch_cap(FastPlan *fp, const Dev &P, const Maps &io, int ring_hi, cudaStream_t st, int *launches) {
    *launches = 0;
    if (!fp) return cudaErrorInvalidValue;
    const int N = P.nside;
    const int s_lo = fp->polar + 1, s_hi = std::min(ring_hi, 2 * N);
    if (s_lo > s_hi) return cudaSuccess;
    cudaError_t e = cudaSuccess;
    auto it = fp->caps.find(s_hi);
    if (it == fp->caps.end()) {
        // shape: as the 8-image instances of sc_convolve (two staged planes per position)
        struct Cand { int threads, R; };
        std::vector<Cand> cands;
        if (fp->mean_nb <= 700.0) cands = {{384, 4}, {256, 4}, {128, 2}};
        else cands = {{256, 4}, {128, 2}};
        const int Lmax = (int)(((size_t)fp->smem_optin - 512 - fp->tab_bytes) / ((size_t)kSymBufH * 2 * 16)) & ~7;
        std::vector<SymTile> tiles;
        FastCfg c;
        for (const Cand &cd : cands) {
            const int W = cd.threads / 32, C = 32 * cd.R;
            for (int shrink = 0; shrink <= W * C / 4 && !c.ok; shrink += 16) {
                tiles.clear();
                const int Lneed = build_sym_tiles(*fp->geo, cd.R, W, W * C - shrink, Lmax, s_hi, s_lo, true, tiles, true, 32, 0, 0, true);
                const size_t smem = fp->tab_bytes + (size_t)kSymBufH * 2 * Lneed * 16;
                if (smem + 512 > (size_t)fp->smem_optin) continue;
                c.threads = cd.threads; c.R = cd.R; c.run = W * C - shrink; c.mirror = true; c.Ltot = Lneed; c.smem = smem;
                c.tot = cd.threads != 384; c.tmem = false; c.ntiles = (int)tiles.size();
                c.ok = true;
            }
            if (c.ok) break;
        }
        if (!c.ok) return cudaErrorInvalidValue;
        if ((e = cudaMalloc((void **)&c.tiles, std::max<size_t>(tiles.size(), 1) * sizeof(SymTile))) != cudaSuccess) return e;
        if (!tiles.empty() && (e = cudaMemcpy(c.tiles, tiles.data(), tiles.size() * sizeof(SymTile), cudaMemcpyHostToDevice)) != cudaSuccess) return e;
        it = fp->caps.emplace(s_hi, c).first;
    }
    const FastCfg &c = it->second;
    if (c.ntiles > 0) {
        if ((e = dispatch_sym(fp, c, P, io, 1, st, c.tiles, c.ntiles, false)) != cudaSuccess) return e;
        ++*launches;
    }
    return e;
}

// latitude chunks for the pipelined host entry: kind 0 = sym kernel, 1 = belt kernel
int fast_chunk_count(const FastPlan *fp, int B, int kind) {
    if (!fp || B < 1 || B > kMaxB || !fp->cfg[B].ok) return 0;
    return kind == 0 ? (int)fp->cfg[B].ch_lo.size() : (fp->belt_ok ? (int)fp->bch_lo.size() : 0);
}
void fast_chunk_rings(const FastPlan *fp, int B, int kind, int i, int *lo, int *hi) {
    if (kind == 0) { *lo = fp->cfg[B].ch_lo[i]; *hi = fp->cfg[B].ch_hi[i]; }
    else { *lo = fp->bch_lo[i]; *hi = fp->bch_hi[i]; }
}

cudaError_t fast_convolve(FastPlan *fp, const Dev &P, const Maps &io, int B, cudaStream_t st, int *launches,
                          cudaEvent_t *ev) {
    int n1 = 0, n2 = 0;
    cudaError_t e;
    if (!ev && fp && B >= 1 && B <= kMaxB && fp->cfg[B].ok && !fp->cfg[B].pair && fp->belt_ok &&
        !std::getenv("SC_NO_OVERLAP")) {
        // Belt kernel first, then the sym kernel launched so that its CTAs may start on the SMs that the belt kernel's
        // CTAs have left (the two write disjoint pixels and read only the inputs): the sym kernel takes its tiles
        // dynamically, so the belt kernel's uneven end is filled.  The tile counter is zeroed before both.
        // (measured: -1 to -2 % at configs 3-5, -0.3 % at the paper-scale config 6).
        const FastCfg &c = fp->cfg[B];
        if ((e = cudaMemsetAsync(fp->tile_ctr, 0, sizeof(int), st)) != cudaSuccess) return e;
        if ((e = fast_launch(fp, P, io, B, 2, st, &n2, -1)) != cudaSuccess) return e;
        if (c.ntiles > 0) {
            if ((e = dispatch_sym(fp, c, P, io, B, st, c.tiles, c.ntiles, true, true)) != cudaSuccess) return e;
            n1 = 1;
        }
        *launches = n1 + n2;
        return cudaSuccess;
    }
    e = fast_launch(fp, P, io, B, 1, st, &n1, -1);
    *launches = n1;
    if (e != cudaSuccess) return e;
    if (ev && (e = cudaEventRecord(ev[0], st)) != cudaSuccess) return e;      // end of the sym kernel
    e = fast_launch(fp, P, io, B, 2, st, &n2, -1);
    *launches += n2;
    if (ev && e == cudaSuccess) e = cudaEventRecord(ev[1], st);              // end of the belt kernel
    return e;
}

int fast_first_belt_ring(const FastPlan *fp) { return fp->first_belt; }

bool fast_available(const FastPlan *fp, int B) { return fp && B >= 1 && B <= kMaxB && fp->cfg[B].ok; }

void fast_plan_destroy(FastPlan *fp) {
    if (!fp) return;
    cudaFree(fp->pairs); cudaFree(fp->pair_off);
    for (auto &c : fp->cfg) {
        cudaFree(c.tiles);
        for (auto &kv : c.band_tiles) cudaFree(kv.second.first);
    }
    for (auto &kv : fp->caps) cudaFree(kv.second.tiles);
    cudaFree(fp->woff); cudaFree(fp->belt_tiles); cudaFree(fp->grp_off); cudaFree(fp->grp_e); cudaFree(fp->tile_ctr); cudaFree(fp->pairsd);
    delete fp;
}

static int env_int(const char *name, int dflt) {
    const char *e = std::getenv(name);
    return e && *e ? std::atoi(e) : dflt;
}

FastPlan *fast_plan_create(const Dev &P, const std::vector<double> &z, const std::vector<double> &s,
                           int max_batch, int *polar_rings, cudaError_t *err) {
    *err = cudaSuccess;
    *polar_rings = 0;
    const int N = P.nside, nr = 4 * N - 1;
    constexpr int Rmax = 4;                        // windows are sized for up to 4 base pixels per thread
    int dev = 0, smem_optin = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int ntab_s = P.ntab;                     // the cells and the one zero cell after them (indices are clamped)
    const size_t tab_bytes = ((size_t)ntab_s * 8 + 127) & ~(size_t)127;
    if (tab_bytes + 8192 > (size_t)smem_optin) return nullptr;       // table does not fit: generic only

    auto ipof = [&](int r) { return r < N ? r : (r <= 3 * N ? N : 4 * N - r); };
    auto shof = [&](int r) { return (r >= N && r <= 3 * N) ? ((r - N) & 1) : 0; };
    auto startof = [&](int r) -> int {
        if (r < N) return 2 * r * (r - 1);
        if (r <= 3 * N) return 2 * N * (N - 1) + (r - N) * 4 * N;
        const int m = 4 * N - r;
        return 12 * N * N - 2 * m * (m + 1);
    };
    const double tmax = (double)(P.ntab - 1);
    // largest |d| for which the 4-term polynomial of 1 - cos d is good to 0.004 table cells: the next term is
    // B scale d^10 / 3628800 with B scale <= 2 tmax / d^2 for a pair inside the disc
    const double dmax = std::min(0.9, std::pow(0.004 * 1814400.0 / tmax, 1.0 / 8.0));

    std::vector<PairEnt> pairs;
    std::vector<int> pair_off(1, 0);
    std::vector<char> eligible(2 * N + 1, 0);
    std::vector<std::vector<PairEnt>> per_ring(2 * N + 1);
    for (int r = 1; r <= 2 * N; ++r) {
        const int ip = ipof(r);
        bool ok = true;
        std::vector<PairEnt> &lst = per_ring[r];
        // walk outwards from r in both directions while rings can hold a neighbour
        auto consider = [&](int rq) -> bool {
            double A64 = 1.0 - (z[r - 1] * z[rq - 1] + s[r - 1] * s[rq - 1]);
            if (A64 < 0) A64 = 0;
            const double Bs = s[r - 1] * s[rq - 1] * P.scale;
            const double wmax = (tmax + 2.0 * (double)P.eps + 0.01 - A64 * P.scale) / Bs;
            if (wmax < 0) return false;
            const int ipq = ipof(rq);
            const double dphi = 2.0 * M_PI / (4.0 * ipq);
            const double H = wmax >= 2.0 ? M_PI : 2.0 * std::asin(std::sqrt(0.5 * wmax));
            const double rho1 = std::fabs(1.0 - (double)ipq / ip);
            const int hw = (int)std::floor(H / dphi + 0.5 + rho1 * (Rmax - 1) + 1e-6);
            if ((hw + 1 + Rmax) * dphi > dmax) ok = false;
            PairEnt e;
            e.A = (float)(A64 * P.scale - 0.5);
            e.c1 = (float)(Bs / 2.0); e.c2 = (float)(-Bs / 24.0); e.c3 = (float)(Bs / 720.0); e.c4 = (float)(-Bs / 40320.0);
            // lane skew of the planar and batch sym instances (at most 3 base pixels per lane): drift of 32 lanes against this ring, + 1;
            // not worth it beyond 8 positions (rings next to the pole), not possible if the longer window would wrap
            e.ex = ipq == ip ? 0 : (int)std::ceil(31.0 * 3.0 * rho1) + 1;
            if (e.ex > 8 || ipq + 2 * hw + 2 * Rmax + 4 + 2 * e.ex >= 4 * ipq) e.ex = 0;
            e.dphi = (float)dphi;
            e.cdc = (float)(M_PI / (4.0 * (double)ip * (double)ipq));
            e.rq = rq; e.hw = hw; e.ipq = ipq; e.shq = shof(rq);
            e.start_n = startof(rq); e.start_s = startof(4 * N - rq);
            lst.push_back(e);
            return true;
        };
        for (int rq = r; rq >= 1; --rq) if (!consider(rq)) break;
        std::reverse(lst.begin(), lst.end());
        for (int rq = r + 1; rq <= nr; ++rq) if (!consider(rq)) break;
        // the window of a whole quadrant must not wrap onto itself
        for (const PairEnt &e : lst) if (e.ipq + 2 * e.hw + 2 * Rmax + 4 >= 4 * e.ipq) ok = false;
        eligible[r] = ok;
    }
    int polar = 0;
    for (int r = 1; r <= 2 * N; ++r) if (!eligible[r]) polar = r;
    if (polar >= 2 * N) return nullptr;                            // nothing for the fast kernel
    // slots: base rings polar+1 .. 2N
    std::vector<int> slot_of(2 * N + 1, -1);
    for (int r = polar + 1; r <= 2 * N; ++r) {
        slot_of[r] = (int)pair_off.size() - 1;
        pairs.insert(pairs.end(), per_ring[r].begin(), per_ring[r].end());
        pair_off.push_back((int)pairs.size());
    }

    FastPlan *fp = new FastPlan;
    fp->geo = std::make_shared<HostGeo>();
    fp->ntab_s = ntab_s; fp->polar = polar; fp->nsm = nsm;
    fp->tab_bytes = tab_bytes; fp->smem_optin = smem_optin;
    fp->mean_nb = 0.5 * (double)P.npix * ((double)P.tmax / P.scale);
    auto fail = [&](cudaError_t e) { *err = e; fast_plan_destroy(fp); return (FastPlan *)nullptr; };
    cudaError_t e;
    if ((e = cudaMalloc((void **)&fp->pairs, std::max<size_t>(pairs.size(), 1) * sizeof(PairEnt))) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc((void **)&fp->pair_off, pair_off.size() * sizeof(int))) != cudaSuccess) return fail(e);
    if ((e = cudaMalloc((void **)&fp->tile_ctr, 64)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpy(fp->pairs, pairs.data(), pairs.size() * sizeof(PairEnt), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
    if ((e = cudaMemcpy(fp->pair_off, pair_off.data(), pair_off.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);

    // ---- belt kernel: base rings whose input rings all have 4N pixels ------------------------------
    std::vector<char> is_belt(2 * N + 1, 0);
    const bool no_belt = std::getenv("SC_NO_BELT") != nullptr;
    // variants (consumer threads, slack floats per plane): tile = 4 x threads base pixels, must divide N
    struct BeltVar { int nc, slack; };
    std::vector<BeltVar> bvars;
    {
        const double mean_nb_b = 0.5 * (double)P.npix * ((double)P.tmax / P.scale);
        if (N % 2048 == 0 && mean_nb_b <= 700.0 && !std::getenv("SC_BELT_NO512")) bvars.push_back({512, 64});
        if (N % 2048 == 0 && mean_nb_b > 700.0 && !std::getenv("SC_BELT_NOTMEM")) { bvars.push_back({512, 256}); bvars.push_back({512, 512}); }
        if (N % 1024 == 0) { bvars.push_back({256, 256}); bvars.push_back({256, 512}); }
        else if (N % 512 == 0) bvars.push_back({128, 256});
    }
    const int bpx = std::getenv("SC_BELT_PX4") ? 4 : 8;                   // pixels per consumer thread
    for (const BeltVar &bv : bvars) {
        if (no_belt || fp->belt_ok) break;
        const int bNC = bv.nc;
        const int T = 4 * bNC;
        std::vector<int> woff(pairs.size(), 0);
        std::vector<int4> btiles;
        int pw_max = 0, ne_max = 0;
        bool fits = true;
        // The input rings of a base ring are cut into groups whose tap arrays fit one tap buffer (a few
        // hundred rings of a few hundred taps for paper-scale discs do not fit as a whole).
        const int kTapCap = 2048, kGroupRings = 96;                       // float2 entries, rings per group
        std::vector<int> grp_off(1, 0), grp_e;
        std::fill(is_belt.begin(), is_belt.end(), 0);
        for (int r = polar + 1; r <= 2 * N; ++r) {                           // slots run over base rings polar+1 .. 2N
            bool all = ipof(r) == N;
            for (const PairEnt &pe : per_ring[r]) if (pe.ipq != N) { all = false; break; }
            is_belt[r] = all;
            const int base = pair_off[slot_of[r]];
            int off = 0, cnt = 0;
            grp_e.push_back(0);
            for (size_t i = 0; i < per_ring[r].size(); ++i) {
                const int ng_max = (2 * per_ring[r][i].hw + bpx + 3 + 3) >> 2; // chunks of 4 staged positions
                const int len = (4 * ng_max + bpx - 2 + 1) & ~1;               // tap pairs, even count
                if (all && (4 * ng_max > bv.slack + bpx || len > kTapCap)) fits = false;   // plane = T - px + 4 ng floats
                if (cnt > 0 && (off + len > kTapCap || cnt >= kGroupRings)) {  // next group
                    grp_e.push_back((int)i); off = 0; cnt = 0;
                }
                woff[base + i] = off;
                off += len; ++cnt;
                if (all) { pw_max = std::max(pw_max, off); ne_max = std::max(ne_max, cnt); }
            }
            grp_e.push_back((int)per_ring[r].size());
            grp_off.push_back((int)grp_e.size());
        }
        for (int r = 2 * N; r > polar; --r) {
            if (!is_belt[r]) { for (int q = r; q > polar; --q) is_belt[q] = 0; break; }   // belt rings are contiguous from 2N down
            for (int k0 = 0; k0 < N; k0 += T) btiles.push_back(make_int4(r, k0, slot_of[r], (int)per_ring[r].size()));
        }
        int nbuf = 0, ntb = 0;
        size_t bsmem = 0;
        if (fits && !btiles.empty()) {
            const int combos[6][2] = {{2, 4}, {2, 3}, {1, 4}, {2, 2}, {1, 3}, {1, 2}};       // (tap buffers, stage buffers)
            for (const auto &cb : combos) {
                bsmem = belt_smem_bytes(bNC, bv.slack, bpx, cb[1], cb[0], pw_max, ne_max);
                if (bsmem + 2048 <= (size_t)smem_optin) { ntb = cb[0]; nbuf = cb[1]; break; }
            }
        }
        if (nbuf >= ((bNC == 512 && bv.slack == 64) ? 3 : 2)) {
            if ((e = cudaMalloc((void **)&fp->woff, woff.size() * sizeof(int))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(fp->woff, woff.data(), woff.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            if ((e = cudaMalloc((void **)&fp->belt_tiles, btiles.size() * sizeof(int4))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(fp->belt_tiles, btiles.data(), btiles.size() * sizeof(int4), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            if ((e = cudaMalloc((void **)&fp->grp_off, grp_off.size() * sizeof(int))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(fp->grp_off, grp_off.data(), grp_off.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            if ((e = cudaMalloc((void **)&fp->grp_e, grp_e.size() * sizeof(int))) != cudaSuccess) return fail(e);
            if ((e = cudaMemcpy(fp->grp_e, grp_e.data(), grp_e.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            fp->belt = BeltDev{fp->pairs, fp->pair_off, fp->woff, fp->belt_tiles, fp->grp_off, fp->grp_e, (int)btiles.size(), pw_max, ne_max, nbuf, ntb, nullptr};
            fp->belt_slack = bv.slack; fp->belt_px = bpx;
            fp->belt_threads = bNC; fp->belt_smem = bsmem; fp->belt_ok = true; fp->belt_tiles_per_ring = N / T;
            // latitude chunks: the tile list runs from ring 2N down to the first belt ring, N / T tiles per ring
            {
                int r_first = 2 * N + 1;
                for (int r = 2 * N; r > polar && is_belt[r]; --r) r_first = r;
                const int nrings = 2 * N - r_first + 1, per_ring_tiles = N / T;
                fp->bch_off.assign(1, 0); fp->bch_lo.clear(); fp->bch_hi.clear();
                int hi = 2 * N;
                const int nbch = std::max(1, env_int("SC_BELT_CHUNKS", kBeltChunksDflt));
                for (int cidx = 1; cidx <= nbch && hi >= r_first; ++cidx) {
                    int lo = 2 * N + 1 - (int)((long long)nrings * cidx / nbch);
                    if (cidx == nbch) lo = r_first;
                    if (lo > hi) continue;
                    fp->bch_lo.push_back(lo); fp->bch_hi.push_back(hi);
                    fp->bch_off.push_back((2 * N - lo + 1) * per_ring_tiles);
                    hi = lo - 1;
                }
            }
        } else {
            std::fill(is_belt.begin(), is_belt.end(), 0);
        }
    }

    // ---- step order of the sym kernel: a step's pair loop takes time ~ the ring's half window, its staging a constant
    // (the whole run), so the rings at the edge of the disc are short steps in which the consumers outrun the producers.
    // Alternate long and short steps (the two stage buffers then average over a pair) instead of walking the rings from
    // north to south.  Belt rings keep their order (tap groups of the belt kernel).
    if (!std::getenv("SC_SYM_RINGORDER")) {
        for (int r = polar + 1; r <= 2 * N; ++r) {
            if (is_belt[r]) continue;
            std::vector<PairEnt> &lst = per_ring[r];
            std::vector<int> idx(lst.size());
            for (size_t i = 0; i < idx.size(); ++i) idx[i] = (int)i;
            std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return lst[a].hw > lst[b].hw; });
            std::vector<PairEnt> out;
            out.reserve(lst.size());
            for (size_t lo = 0, hi = idx.size(); lo < hi;) {
                out.push_back(lst[idx[lo++]]);
                if (lo < hi) out.push_back(lst[idx[--hi]]);
            }
            lst = out;
            std::copy(lst.begin(), lst.end(), pairs.begin() + pair_off[slot_of[r]]);
        }
        if ((e = cudaMemcpy(fp->pairs, pairs.data(), pairs.size() * sizeof(PairEnt), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
    }

    // ---- fp64 ring pairs for plans with steep tables (Dev::hp), in the final order of `pairs` ------------------------
    if (P.hp) {
        std::vector<PairEntD> pd(pairs.size());
        for (int r = polar + 1; r <= 2 * N; ++r) {
            const int base = pair_off[slot_of[r]];
            for (size_t i = 0; i < per_ring[r].size(); ++i) {
                const int rq = per_ring[r][i].rq;
                double A64 = 1.0 - (z[r - 1] * z[rq - 1] + s[r - 1] * s[rq - 1]);
                if (A64 < 0) A64 = 0;
                pd[base + i] = PairEntD{A64 * P.scale, s[r - 1] * s[rq - 1] * P.scale, 2.0 * M_PI / (4.0 * ipof(rq)),
                                        M_PI / (4.0 * (double)ipof(r) * (double)ipof(rq))};
            }
        }
        if ((e = cudaMalloc((void **)&fp->pairsd, std::max<size_t>(pd.size(), 1) * sizeof(PairEntD))) != cudaSuccess) return fail(e);
        if ((e = cudaMemcpy(fp->pairsd, pd.data(), pd.size() * sizeof(PairEntD), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
        if (fp->belt_ok) fp->belt.pairsd = fp->pairsd;
    }

    // ---- sym kernel: per batch size pick (threads, R) so that table + double-buffered stage fit ------
    // Tiles are packed from sub-tiles (runs of base pixels on one ring, 32 R pixels per warp): whole
    // CTA-wide runs first, the ragged remainders of all rings are bin-packed (first fit, decreasing).
    (void)max_batch;
    struct Cand { int threads, R; bool mirror; bool pair = false; bool planar = false; };
    for (int B = 1; B <= kMaxB; ++B) {
        FastCfg &c = fp->cfg[B];
        std::vector<Cand> cands;
        // 384 consumer threads only come without the second accumulator set (registers): plain fp32
        // running sums, good to ~3e-7 relative rms for discs of a few hundred pixels (measured 2.7e-7 at
        // 425), so only while the mean disc holds at most 700 pixels (4.7e-7 measured at 1380 for a Gaussian, 6.9e-7 at 960 for a cancelling split kernel)
        const double mean_nb = 0.5 * (double)P.npix * ((double)P.tmax / P.scale);
        // between 700 and 6000 pixels per disc the 384-consumer variant keeps the running totals in tensor memory
        // (4-6 % faster than 256 consumers with both sets in registers; slower again for still larger discs)
        if (B == 1 && (mean_nb <= 700.0 || (mean_nb <= 6000.0 && !std::getenv("SC_SYM_NOTMEM")))) cands = {{384, 4, false}, {256, 4, false}, {256, 2, false}, {128, 2, false}};
        else if (B == 1) cands = {{256, 4, false}, {256, 2, false}, {128, 2, false}};
        else cands = {{256, 2, false}, {128, 2, false}, {128, 1, false}};
        // one map per launch: 16 images per pair geometry (mirror symmetry as well) -- half the table gathers and
        // geometry per pair; twice the staged bytes per base pixel, so 192 consumer threads x 4 base pixels
        if (B == 1 && !std::getenv("SC_SYM_NOMIRROR")) cands.insert(cands.begin(), Cand{192, 4, true});
        // ... or 256 consumer threads x 3 base pixels: the same 768-pixel tiles with 8 consumer warps
        if (B == 1 && !std::getenv("SC_SYM_NOMIRROR") && !std::getenv("SC_SYM_NOR3")) cands.insert(cands.begin(), Cand{256, 3, true});
        // ... with planar staging (one plane per image, TMA bulk copies, lane skew; sc_sym_pl.cu) when the planes fit next to
        // the table, for discs of at most 2500 pixels (measured, sym kernel: config 3 -10 %, config 4 -10 %; with the
        // tensor-memory totals of larger discs Nside 2048 35' -2.6 %, Nside 1024 72' -2 %, Nside 2048 60' +0.3 %) and for maps
        // with at least one full tile per SM (config 1: 0.031 against 0.022 ms, 64 tiny bulk copies per step)
        if (B == 1 && !std::getenv("SC_SYM_NOMIRROR") && !std::getenv("SC_SYM_NOR3") && !std::getenv("SC_SYM_NOPLANAR") && mean_nb <= 2500.0 &&
            tab_bytes + (size_t)kSymBufH * 16 * kPlanarPlane * 4 + 512 <= (size_t)smem_optin)
            cands.insert(cands.begin(), Cand{256, 3, true, false, true});
        // ... and as lane pairs (sc_sym_pair.cu): 32 accumulators per lane, 12 (small discs) or 8 consumer warps
        if (B == 1 && !std::getenv("SC_SYM_NOMIRROR") && std::getenv("SC_SYM_PAIR"))
            cands.insert(cands.begin(), mean_nb <= 700.0 ? Cand{env_int("SC_PAIR_NC", 384), 4, true, true} : Cand{256, 4, true, true});
        if (P.hp) {                                         // fp64 table coordinate: the 16-image instance only, one map per launch
            if (B > 1) continue;
            cands = {Cand{256, 3, true}, Cand{192, 4, true}, Cand{256, 4, false}, Cand{256, 2, false}, Cand{128, 2, false}};
        }
        const int fr = env_int("SC_SYM_R", 0), ft = env_int("SC_SYM_THREADS", 0);
        if (!P.hp && fr > 0 && ft > 0 && (fr == 1 || fr == 2 || (fr == 4 && B <= 2)) && (ft == 128 || ft == 256 || (ft == 384 && fr == 4 && B == 1)))
            cands.insert(cands.begin(), Cand{ft, fr, false});
        for (const Cand &cd : cands) {
            const int R = cd.R, W = cd.threads / 32, C = (cd.pair ? 16 : 32) * R;
            // full-width runs may be a little shorter than the CTA (last lanes idle) if that makes the
            // staged runs fit into shared memory
            // small maps: fewer full-width tiles than SMs -> shorter runs (idle lanes, but every SM gets a tile)
            int shrink0 = 0;
            if (B == 1 && !std::getenv("SC_SYM_NOSPREAD")) {
                long long base_px = 0;
                for (int r = polar + 1; r <= 2 * N; ++r)
                    if (!is_belt[r]) base_px += cd.mirror ? (ipof(r) + 2) / 2 : ipof(r);
                const long long n0 = (base_px + W * C - 1) / (W * C);
                if (n0 < fp->nsm) {
                    const int want = std::max(2 * C, (int)(((base_px + fp->nsm - 1) / fp->nsm + 31) / 32) * 32);
                    if (want < W * C) shrink0 = (W * C - want) & ~15;
                }
            }
            if (cd.planar && shrink0 > 0) continue;
            for (int shrink = shrink0; shrink <= std::max(W * C / 4, shrink0) && !c.ok; shrink += 16) {
            const int run = W * C - shrink;
            // a tile holds at most W warps, kMaxSub runs and Lmax staged positions (shared memory)
            const int npl = cd.mirror ? 4 : 2;                      // staged planes per position (float4 of rotation images each)
            const size_t stat = cd.pair ? 3072 : 512;            // static shared memory of the kernel (barriers; step records)
            const int Lmax = cd.planar ? kPlanarPlane : (int)(((size_t)smem_optin - stat - tab_bytes) / ((size_t)kSymBufH * B * npl * 16)) & ~7;
            HostGeo &g = *fp->geo;
            g.N = N; g.polar = polar; g.per_ring = per_ring; g.slot_of = slot_of; g.pair_off = pair_off; g.is_belt = is_belt;
            auto build = [&](int r_hi, int r_lo, std::vector<SymTile> &tl) { return build_sym_tiles(g, R, W, run, Lmax, r_hi, r_lo, cd.mirror, tl, false, cd.pair ? 16 : 32, shrink0 > 0 ? (run + C - 1) / C : 0, cd.planar ? kPlanarPad : 0, true); };
            // (1) the whole range in one work-sorted list: sc_convolve; (2) the same rings in kSymChunks
            // latitude chunks from the belt towards the pole, each sorted: the pipelined host entry
            std::vector<SymTile> tiles;
            int Ltot = build(2 * N, polar + 1, tiles);
            int sym_hi = 2 * N;
            while (sym_hi > polar && is_belt[sym_hi]) --sym_hi;
            std::vector<int> ch_off(1, (int)tiles.size()), ch_lo, ch_hi;
            {
                const long long nsymch = std::max(1, env_int("SC_SYM_CHUNKS", kSymChunksDflt));
                long long total_px = 0, acc_px = 0;
                for (int r = sym_hi; r > polar; --r) total_px += ipof(r);
                int hi = sym_hi, nch = 0;
                for (int r = sym_hi; r > polar; --r) {
                    acc_px += ipof(r);
                    if (r == polar + 1 || acc_px * nsymch >= total_px * (nch + 1)) {
                        Ltot = std::max(Ltot, build(hi, r, tiles));
                        ch_off.push_back((int)tiles.size()); ch_lo.push_back(r); ch_hi.push_back(hi);
                        hi = r - 1; ++nch;
                    }
                }
            }
            if (cd.planar && Ltot > kPlanarPlane) continue;
            if (cd.planar) Ltot = kPlanarPlane;                   // the planar instances' plane length is a compile-time constant
            const size_t smem = tab_bytes + (size_t)kSymBufH * B * npl * Ltot * 16;
            if (smem + stat > (size_t)smem_optin) continue;
            c.ntiles_all = ch_off[0]; c.ch_off = ch_off; c.ch_lo = ch_lo; c.ch_hi = ch_hi;
            c.threads = cd.threads; c.R = R; c.Ltot = Ltot; c.smem = smem; c.ntiles = c.ntiles_all; c.run = run;
            c.mirror = cd.mirror; c.pair = cd.pair; c.planar = cd.planar; c.skew = true;
            c.tmem = !cd.pair && (B == 1 && (cd.threads == 384 || cd.mirror) && mean_nb > 700.0);      // large discs: two-level sums, totals in TMEM
            // a single accumulator set (plain fp32 running sums) only for one map and discs of at most 700 pixels
            c.tot = !(B == 1 && (cd.threads == 384 || cd.mirror) && mean_nb <= 700.0);
            if (cd.pair) c.tot = mean_nb > 700.0;
            if ((e = cudaMalloc((void **)&c.tiles, std::max<size_t>(tiles.size(), 1) * sizeof(SymTile))) != cudaSuccess) return fail(e);
            if (!tiles.empty() && (e = cudaMemcpy(c.tiles, tiles.data(), tiles.size() * sizeof(SymTile), cudaMemcpyHostToDevice)) != cudaSuccess) return fail(e);
            c.ok = true;
            }
            if (c.ok) break;
        }
    }
    fp->first_belt = 2 * N + 1;
    for (int r = 2 * N; r > polar && is_belt[r]; --r) fp->first_belt = r;
    *polar_rings = polar;
    return fp;
}

}  // namespace sc
