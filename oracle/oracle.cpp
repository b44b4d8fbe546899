/*
 * oracle/oracle.cpp -- THE ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, single-threaded CPU implementation of the track-repeating hot path of
 * Yepes, Mirkovic & Taddei, written step by step from DESIGN.md §3
 * (rules R1-R9, which restate SURVEY.md §8(c) O1-O9).  It shares no code with
 * paper_1011_2188_b200/csrc/ and is only ever used by tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1 conservation, P2 water identity vs an
 * independent Siddon voxelisation, P3 range scaling, P4 brute-force f64 walker, P5 DB closed
 * forms, P6 Philox known answers, P7 linearity, P8 DDA bookkeeping, P9 sampler moments, P10 slab
 * consistency.  PARITY UNPINNED: agreement with GEANT4 / CPU FDC / the patient case
 * -- that data does not exist here.
 *
 * Real type: `float` is the arithmetic contract (compile with
 * -ffp-contract=off); `double` runs the same rules in f64 for error bounding.
 */
#include <cstdint>
#include <cmath>
#include <cstring>
#include <limits>
#include <vector>
#include <algorithm>
#include <utility>

namespace {

/* ---------------------------------------------------------------- R3: Philox4x32-10 */
struct Block { uint32_t w[4]; };

Block philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
    for (int round = 0; round < 10; ++round) {
        uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(prod0 >> 32), lo0 = (uint32_t)prod0;
        uint32_t hi1 = (uint32_t)(prod1 >> 32), lo1 = (uint32_t)prod1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    Block b; b.w[0] = c0; b.w[1] = c1; b.w[2] = c2; b.w[3] = c3;
    return b;
}

/* R3: signed(x) = (f32(x>>9) + 0.5) * 2^-22 - 1, exact in f32 */
float signed_unit(uint32_t x) { return ((float)(x >> 9) + 0.5f) * 2.384185791015625e-07f - 1.0f; }

/* ---------------------------------------------------------------- R5: fixed-order ln, f64 */
double contract_ln(double x)
{
    uint64_t bits; std::memcpy(&bits, &x, 8);
    int e = (int)((bits >> 52) & 0x7ff) - 1022;
    bits = (bits & 0x000fffffffffffffULL) | 0x3fe0000000000000ULL;
    double m; std::memcpy(&m, &bits, 8);
    if (m < 0.70710678118654757) { m = m * 2.0; e = e - 1; }
    double z = (m - 1.0) / (m + 1.0);
    double q = z * z;
    double S = 1.0 / 29.0;
    for (int n = 13; n >= 0; --n) S = std::fma(S, q, 1.0 / (double)(2 * n + 1));
    return std::fma((double)e, 0.6931471805599453, (2.0 * z) * S);
}

/* ---------------------------------------------------------------- small helpers */
template <class T> T FMA(T a, T b, T c) { return std::fma(a, b, c); }
template <class T> T dot3(const T *a, const T *b) { return FMA(a[2], b[2], FMA(a[1], b[1], a[0] * b[0])); }

struct Knot { float hu, rho, s, t; };

struct Beamlet {
    float origin[3], e1[3], e2[3], dir[3];
    float energy, spot_u, spot_v, sigma;
    uint64_t n_protons;
};

struct Stats {
    uint64_t protons, proton_steps, deposits, missed, escaped, stopped, grid_sum, q_replayed, q_escaped;
};

struct TrackDB {
    const float *dx, *dy, *dz, *dE, *E;
    uint64_t n_steps;
    const uint64_t *track_off; uint32_t n_tracks;
    const uint32_t *bin_first; uint32_t n_bins;
    float e_min, e_bin;
};

const int HU_LO = -1024, HU_HI = 3071, N_MAT = 4096;

/* R1 */
void material_lut(const Knot *k, int n, float *rho, float *w, float *fth)
{
    for (int h = HU_LO; h <= HU_HI; ++h) {
        double r, s, t;
        if ((double)h <= (double)k[0].hu) { r = k[0].rho; s = k[0].s; t = k[0].t; }
        else if ((double)h >= (double)k[n - 1].hu) { r = k[n - 1].rho; s = k[n - 1].s; t = k[n - 1].t; }
        else {
            int i = 0;
            while (!((double)k[i].hu <= (double)h && (double)h < (double)k[i + 1].hu)) ++i;
            double frac = ((double)h - (double)k[i].hu) / ((double)k[i + 1].hu - (double)k[i].hu);
            r = (double)k[i].rho + ((double)k[i + 1].rho - (double)k[i].rho) * frac;
            s = (double)k[i].s + ((double)k[i + 1].s - (double)k[i].s) * frac;
            t = (double)k[i].t + ((double)k[i + 1].t - (double)k[i].t) * frac;
        }
        float rf = (float)r, sf = (float)s, tf = (float)t;
        rho[h - HU_LO] = rf;
        w[h - HU_LO] = (float)((double)rf * (double)sf);
        fth[h - HU_LO] = (float)std::sqrt((double)tf / (double)sf);
    }
}

int mat_index(int16_t hu) { int h = hu; if (h < HU_LO) h = HU_LO; if (h > HU_HI) h = HU_HI; return h - HU_LO; }

/* R5: first accepted candidate pair of `purpose`; returns false if 16 attempts all fail */
bool candidate_pair(uint64_t i, uint64_t seed, uint32_t purpose, float &a, float &b, float &r2)
{
    for (uint32_t attempt = 0; attempt < 16; ++attempt) {
        Block B = philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), purpose, attempt,
                                (uint32_t)seed, (uint32_t)(seed >> 32));
        for (int pair = 0; pair < 2; ++pair) {
            a = signed_unit(B.w[2 * pair]);
            b = signed_unit(B.w[2 * pair + 1]);
            r2 = std::fma(a, a, b * b);
            if (r2 > 0.0f && r2 <= 1.0f) return true;
        }
    }
    return false;
}

/* the state a proton starts with after R2-R6 (exposed for the sampler pins) */
template <class T> struct Start {
    uint32_t beamlet, track; uint64_t k0, k_end;
    T p[3], R[3][3]; int iv[3]; int missed;
    float c, s, gx, gy;
};

struct Geometry {
    const int16_t *hu; int n[3]; float sp[3];
    float lut_rho[N_MAT], lut_w[N_MAT], lut_f[N_MAT];
};

/* R4 bin */
int energy_bin(float E0, float e_min, float e_bin)
{
    float x = (E0 - e_min) / e_bin;
    return x <= 0.0f ? 0 : (int)std::ceil(x);
}

template <class T>
int start_from(const Geometry &G, const TrackDB &db, const Beamlet &B, uint64_t i, uint64_t seed, uint32_t flags, Start<T> &S);

/* R2-R6 for proton i.  Returns <0 on FDC_ERANGE-type failure. */
template <class T>
int start_proton(const Geometry &G, const TrackDB &db, const Beamlet *bl, uint32_t n_bl,
                 uint64_t i, uint64_t seed, uint32_t flags, Start<T> &S)
{
    /* R2 */
    uint64_t lo = 0; uint32_t b = 0;
    for (; b < n_bl; ++b) { if (i < lo + bl[b].n_protons) break; lo += bl[b].n_protons; }
    if (b == n_bl) return -1;
    S.beamlet = b;
    return start_from<T>(G, db, bl[b], i, seed, flags, S);
}

/* R12: a phase-space particle (position, unit direction, energy; "phase-space array") is a
 * one-proton beamlet with no lateral spread whose transverse frame is fixed by its direction d:
 * a = the axis with the smallest |d_a| (lowest index on ties), t = e_a - d_a d, e1 = t / |t|, e2 = d x e1. */
struct Particle { float pos[3], dir[3], energy, reserved; };
void frame_rule(const float d[3], float e1[3], float e2[3])
{
    int a = 0;
    if (std::fabs(d[1]) < std::fabs(d[a])) a = 1;
    if (std::fabs(d[2]) < std::fabs(d[a])) a = 2;
    float t[3];
    for (int b = 0; b < 3; ++b) t[b] = std::fma(-d[a], d[b], b == a ? 1.0f : 0.0f);
    const float n2 = std::fma(t[2], t[2], std::fma(t[1], t[1], t[0] * t[0]));
    const float inv = 1.0f / std::sqrt(n2);
    for (int b = 0; b < 3; ++b) e1[b] = t[b] * inv;
    e2[0] = std::fma(d[1], e1[2], -(d[2] * e1[1]));
    e2[1] = std::fma(d[2], e1[0], -(d[0] * e1[2]));
    e2[2] = std::fma(d[0], e1[1], -(d[1] * e1[0]));
}
Beamlet beamlet_of(const Particle &P)
{
    Beamlet B; std::memset(&B, 0, sizeof B);
    for (int a = 0; a < 3; ++a) { B.origin[a] = P.pos[a]; B.dir[a] = P.dir[a]; }
    frame_rule(P.dir, B.e1, B.e2);
    B.energy = P.energy; B.spot_u = 0.0f; B.spot_v = 0.0f; B.sigma = 0.0f; B.n_protons = 1;
    return B;
}

/* R4-R6 for proton i (its random-number identity) started from beamlet B */
template <class T>
int start_from(const Geometry &G, const TrackDB &db, const Beamlet &B, uint64_t i, uint64_t seed, uint32_t flags, Start<T> &S)
{
    /* R4 */
    int beta = energy_bin(B.energy, db.e_min, db.e_bin);
    if (beta >= (int)db.n_bins) return -2;
    uint32_t n_beta = db.bin_first[beta + 1] - db.bin_first[beta];
    if (n_beta == 0) return -2;
    Block B0 = philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), 0u, 0u, (uint32_t)seed, (uint32_t)(seed >> 32));
    uint32_t j = db.bin_first[beta] + (uint32_t)(((uint64_t)B0.w[0] * (uint64_t)n_beta) >> 32);
    S.track = j;
    uint64_t k = db.track_off[j], kend = db.track_off[j + 1];
    while (k < kend && !(db.E[k] <= B.energy)) ++k;
    S.k0 = k; S.k_end = kend;
    /* R5 azimuth */
    float c = 1.0f, s = 0.0f, a, bb, r2;
    if ((flags & 1u) && candidate_pair(i, seed, 1u, a, bb, r2)) {
        c = std::fma(a, a, -(bb * bb)) / r2;
        s = ((a + a) * bb) / r2;
    }
    /* R5 lateral offset */
    float gx = 0.0f, gy = 0.0f;
    if (B.sigma > 0.0f && candidate_pair(i, seed, 2u, a, bb, r2)) {
        double r2d = (double)r2;
        double fac = std::sqrt((-2.0 * contract_ln(r2d)) / r2d);
        gx = (float)((double)B.sigma * ((double)a * fac));
        gy = (float)((double)B.sigma * ((double)bb * fac));
    }
    S.c = c; S.s = s; S.gx = gx; S.gy = gy;
    float u = B.spot_u + gx, v = B.spot_v + gy;
    float pf[3];
    for (int ax = 0; ax < 3; ++ax) {
        pf[ax] = std::fma(v, B.e2[ax], std::fma(u, B.e1[ax], B.origin[ax]));
        S.R[ax][0] = (T)std::fma(s, B.e2[ax], c * B.e1[ax]);
        S.R[ax][1] = (T)std::fma(c, B.e2[ax], (-s) * B.e1[ax]);
        S.R[ax][2] = (T)B.dir[ax];
    }
    /* R14 (flag 32): re-align the sub-track.  A proton that starts at step k0 > first re-uses a track
     * that has already been deflected; with the flag, R0 is followed by the minimal rotation taking the
     * unit direction u of step k0 to the database z axis, so that the first replayed step points along
     * the beam (R u = dir).  Same closed form as the R7 rotation with w' = (0,0,1).  Nothing is done if
     * there is no step to replay, step k0 has zero length, or 1 + u_z < 1e-6. */
    if ((flags & 32u) && S.k0 < S.k_end) {
        const T d[3] = {(T)db.dx[S.k0], (T)db.dy[S.k0], (T)db.dz[S.k0]};
        const T l2 = FMA(d[2], d[2], FMA(d[1], d[1], d[0] * d[0]));
        if (l2 != (T)0) {
            const T il = (T)1 / std::sqrt(l2);
            const T uu[3] = {d[0] * il, d[1] * il, d[2] * il};
            const T wz[3] = {(T)0, (T)0, (T)1};
            const T cc = dot3(uu, wz);
            const T den = (T)1 + cc;
            if (den >= (T)1e-6f) {
                T vv[3];
                vv[0] = FMA(uu[1], wz[2], -(uu[2] * wz[1]));
                vv[1] = FMA(uu[2], wz[0], -(uu[0] * wz[2]));
                vv[2] = FMA(uu[0], wz[1], -(uu[1] * wz[0]));
                const T kk = (T)1 / den;
                const T kv[3] = {kk * vv[0], kk * vv[1], kk * vv[2]};
                T dQ[3][3];
                dQ[0][0] = FMA(kv[0], vv[0], cc); dQ[1][1] = FMA(kv[1], vv[1], cc); dQ[2][2] = FMA(kv[2], vv[2], cc);
                dQ[0][1] = FMA(kv[0], vv[1], -vv[2]); dQ[1][0] = FMA(kv[0], vv[1], vv[2]);
                dQ[0][2] = FMA(kv[0], vv[2], vv[1]);  dQ[2][0] = FMA(kv[0], vv[2], -vv[1]);
                dQ[1][2] = FMA(kv[1], vv[2], -vv[0]); dQ[2][1] = FMA(kv[1], vv[2], vv[0]);
                T Rn[3][3];
                for (int a2 = 0; a2 < 3; ++a2)
                    for (int j2 = 0; j2 < 3; ++j2)
                        Rn[a2][j2] = FMA(S.R[a2][2], dQ[2][j2], FMA(S.R[a2][1], dQ[1][j2], S.R[a2][0] * dQ[0][j2]));
                for (int a2 = 0; a2 < 3; ++a2) for (int j2 = 0; j2 < 3; ++j2) S.R[a2][j2] = Rn[a2][j2];
            }
        }
    }
    /* R6 (always in f32: it only places the start point) */
    float hi[3]; bool inside = true;
    for (int ax = 0; ax < 3; ++ax) {
        hi[ax] = (float)G.n[ax] * G.sp[ax];
        if (!(pf[ax] >= 0.0f && pf[ax] <= hi[ax])) inside = false;
    }
    S.missed = 0;
    int enter_axis = -1;
    if (!inside) {
        const float INF = std::numeric_limits<float>::infinity();
        float t_in = -INF, t_out = INF;
        for (int ax = 0; ax < 3; ++ax) {
            float nr, fr;
            if (B.dir[ax] != 0.0f) {
                float inv = 1.0f / B.dir[ax];
                float t0 = (0.0f - pf[ax]) * inv, t1 = (hi[ax] - pf[ax]) * inv;
                nr = t0 < t1 ? t0 : t1; fr = t0 < t1 ? t1 : t0;
            } else {
                if (pf[ax] < 0.0f || pf[ax] > hi[ax]) { S.missed = 1; }
                nr = -INF; fr = INF;
            }
            if (nr > t_in) { t_in = nr; enter_axis = ax; }
            if (fr < t_out) t_out = fr;
        }
        if (t_in > t_out || t_out < 0.0f) S.missed = 1;
        if (S.missed) return 0;
        for (int ax = 0; ax < 3; ++ax) pf[ax] = std::fma(t_in, B.dir[ax], pf[ax]);
    }
    for (int ax = 0; ax < 3; ++ax) {
        float inv_s = 1.0f / G.sp[ax];
        int idx = (int)std::floor(pf[ax] * inv_s);
        if (idx < 0) idx = 0;
        if (idx > G.n[ax] - 1) idx = G.n[ax] - 1;
        if (ax == enter_axis) idx = B.dir[ax] > 0.0f ? 0 : G.n[ax] - 1;
        S.iv[ax] = idx;
        S.p[ax] = (T)pf[ax];
    }
    return 0;
}

/* optional per-deposit trace for the bookkeeping pins (P8) */
struct Trace { uint64_t *voxel; uint64_t *share; uint32_t *step; uint64_t cap, n; };

/* R10: sum-of-squares tallies ("a second tallying array ... the sum of the squares of the
 * deposited energy", eq. (2)).  Operand e' = e >> 8 (quanta of 2^-16 MeV, clamped to 2^32-1), tally
 * += e'^2 (quanta of 2^-32 MeV^2).
 *   by_history: e = ALL the energy history i left in the voxel -- eq. (2)'s D_i, the plain definition.
 *   by_visit  : e = the energy left during one uninterrupted stay in the voxel (from entering it to
 *               crossing out of it); equal to by_history unless a history re-enters a voxel (reading A23). */
struct Squares { uint64_t *by_visit; uint64_t *by_history; };
uint64_t sq_operand(uint64_t e) { uint64_t x = e >> 8; if (x > 0xffffffffull) x = 0xffffffffull; return x * x; }

typedef std::vector<std::pair<uint64_t, uint64_t>> History;    /* every (voxel, share) of one history */
void reduce_history(History &history, Squares *sq)
{
    if (!(sq && sq->by_history)) return;
    std::sort(history.begin(), history.end());
    for (size_t a = 0; a < history.size();) {
        size_t b = a; uint64_t e = 0;
        while (b < history.size() && history[b].first == history[a].first) { e += history[b].second; ++b; }
        sq->by_history[history[a].first] += sq_operand(e);
        a = b;
    }
}

/* R15: histories with several trajectories ("each history ... the trajectories"; L71 "selecting
 * the trajectory").  Secondaries of track j are sec.track[sec.first[j] .. sec.first[j+1]) (tracks outside every
 * energy bin), each starting where its parent stands at the END of the parent's step number sec.step[] (counted
 * from the parent's first step; ascending within a parent).  A proton that joins the parent at step k0 skips the
 * secondaries that branched before k0; one that escapes before a branch step never starts that secondary. */
struct Secondaries { const uint32_t *first, *track, *step; };

/* R7 + R8 for one trajectory.  spawn: receives the start states of the secondaries whose branch step was completed;
 * secondary: this trajectory is one (its fate is not counted in escaped / stopped); hist: the history's deposit
 * list shared by its trajectories (the caller reduces it), or null for a local one. */
template <class T>
void transport(const Geometry &G, const TrackDB &db, Start<T> &S, uint64_t *grid, Stats &st, Trace *tr,
               T *end_state /* p[3], g[3] of the last step, may be null */, Squares *sq = nullptr,
               const Secondaries *sec = nullptr, std::vector<Start<T>> *spawn = nullptr, bool secondary = false, History *hist = nullptr)
{
    uint64_t visit_vox = 0, visit_sum = 0;                       /* R10 by_visit */
    History local_history;
    History &history = hist ? *hist : local_history;             /* R10 by_history */
    auto end_visit = [&]() { if (sq && sq->by_visit && visit_sum) sq->by_visit[visit_vox] += sq_operand(visit_sum); visit_sum = 0; };
    auto end_history = [&]() { end_visit(); if (!hist) reduce_history(history, sq); };
    const uint64_t track_first = db.track_off[S.track];
    uint32_t s_i = 0, s_end = 0;
    if (sec && spawn) {
        s_i = sec->first[S.track]; s_end = sec->first[S.track + 1];
        while (s_i < s_end && (uint64_t)sec->step[s_i] < S.k0 - track_first) ++s_i;        /* branched before the proton joined */
    }
    const T INF = std::numeric_limits<T>::infinity();
    const T TINY = (T)7.888609052210118e-31;     /* 2^-100 */
    T p[3] = {S.p[0], S.p[1], S.p[2]};
    T R[3][3];
    for (int a = 0; a < 3; ++a) for (int m = 0; m < 3; ++m) R[a][m] = S.R[a][m];
    int iv[3] = {S.iv[0], S.iv[1], S.iv[2]};
    const T sp[3] = {(T)G.sp[0], (T)G.sp[1], (T)G.sp[2]};
    bool have_prev = false; T u_prev[3] = {0, 0, 0};
    T g[3] = {0, 0, 0};

    for (uint64_t k = S.k0; k < S.k_end; ++k) st.q_replayed += (uint64_t)std::llrint(db.dE[k] * 16777216.0f);

    for (uint64_t k = S.k0; k < S.k_end; ++k) {
        st.proton_steps++;
        const uint64_t Q = (uint64_t)std::llrint(db.dE[k] * 16777216.0f);      /* R8 */
        uint64_t vox = (uint64_t)iv[0] + (uint64_t)G.n[0] * ((uint64_t)iv[1] + (uint64_t)G.n[1] * (uint64_t)iv[2]);
        auto deposit = [&](uint64_t v, uint64_t q) {
            if (q == 0) return;
            grid[v] += q; st.deposits++;
            if (sq) { visit_vox = v; visit_sum += q; if (sq->by_history) history.push_back(std::make_pair(v, q)); }
            if (tr && tr->n < tr->cap) { tr->voxel[tr->n] = v; tr->share[tr->n] = q; tr->step[tr->n] = (uint32_t)(k - S.k0); tr->n++; }
        };
        const T d[3] = {(T)db.dx[k], (T)db.dy[k], (T)db.dz[k]};
        const T l2 = FMA(d[2], d[2], FMA(d[1], d[1], d[0] * d[0]));
        auto branch_after = [&](uint64_t kk) {                    /* R15: the parent stands at the end of step kk */
            while (s_i < s_end && (uint64_t)sec->step[s_i] == kk - track_first) {
                Start<T> B; std::memset(&B, 0, sizeof B);
                B.track = sec->track[s_i]; B.k0 = db.track_off[B.track]; B.k_end = db.track_off[B.track + 1];
                for (int a = 0; a < 3; ++a) { B.p[a] = p[a]; B.iv[a] = iv[a]; for (int m = 0; m < 3; ++m) B.R[a][m] = R[a][m]; }
                spawn->push_back(B); ++s_i;
            }
        };
        if (l2 == (T)0) { deposit(vox, Q); branch_after(k); continue; }
        const T l = std::sqrt(l2);
        const T il = (T)1 / l;
        const T u[3] = {d[0] * il, d[1] * il, d[2] * il};

        /* angle */
        if (have_prev) {
            const T f = (T)G.lut_f[mat_index(G.hu[vox])];
            if (f != (T)1) {
                const T c = dot3(u_prev, u);
                if (c > (T)0) {
                    T w[3];
                    for (int a = 0; a < 3; ++a) {
                        T e = FMA(-c, u_prev[a], u[a]);
                        w[a] = FMA(f, e, c * u_prev[a]);
                    }
                    const T nrm = (T)1 / std::sqrt(dot3(w, w));
                    for (int a = 0; a < 3; ++a) w[a] = w[a] * nrm;
                    const T cc = dot3(u, w);
                    const T den = (T)1 + cc;
                    if (den >= (T)1e-6f) {
                        T v[3];
                        v[0] = FMA(u[1], w[2], -(u[2] * w[1]));
                        v[1] = FMA(u[2], w[0], -(u[0] * w[2]));
                        v[2] = FMA(u[0], w[1], -(u[1] * w[0]));
                        const T kk = (T)1 / den;
                        const T kv[3] = {kk * v[0], kk * v[1], kk * v[2]};
                        T dQ[3][3];
                        dQ[0][0] = FMA(kv[0], v[0], cc);
                        dQ[1][1] = FMA(kv[1], v[1], cc);
                        dQ[2][2] = FMA(kv[2], v[2], cc);
                        dQ[0][1] = FMA(kv[0], v[1], -v[2]);
                        dQ[1][0] = FMA(kv[0], v[1], v[2]);
                        dQ[0][2] = FMA(kv[0], v[2], v[1]);
                        dQ[2][0] = FMA(kv[0], v[2], -v[1]);
                        dQ[1][2] = FMA(kv[1], v[2], -v[0]);
                        dQ[2][1] = FMA(kv[1], v[2], v[0]);
                        T Rn[3][3];
                        for (int a = 0; a < 3; ++a)
                            for (int j = 0; j < 3; ++j)
                                Rn[a][j] = FMA(R[a][2], dQ[2][j], FMA(R[a][1], dQ[1][j], R[a][0] * dQ[0][j]));
                        for (int a = 0; a < 3; ++a) for (int j = 0; j < 3; ++j) R[a][j] = Rn[a][j];
                    }
                }
            }
        }
        u_prev[0] = u[0]; u_prev[1] = u[1]; u_prev[2] = u[2]; have_prev = true;

        /* direction in the phantom */
        for (int a = 0; a < 3; ++a) g[a] = FMA(R[a][2], u[2], FMA(R[a][1], u[1], R[a][0] * u[0]));

        /* voxel walk */
        T tMax[3], tDelta[3]; int dirn[3];
        for (int a = 0; a < 3; ++a) {
            if (std::fabs(g[a]) < TINY) { tMax[a] = INF; tDelta[a] = INF; dirn[a] = 0; }
            else {
                T inv = (T)1 / g[a];
                T face = g[a] > (T)0 ? (T)(iv[a] + 1) * sp[a] : (T)(iv[a]) * sp[a];
                tMax[a] = std::fmax((T)0, (face - p[a]) * inv);
                tDelta[a] = std::fabs(sp[a] * inv);
                dirn[a] = g[a] > (T)0 ? 1 : -1;
            }
        }
        T t_cur = 0, l_rem = l, acc = 0, t_end = 0;
        uint64_t q_done = 0;
        bool escaped = false;
        for (;;) {
            const T w = (T)G.lut_w[mat_index(G.hu[vox])];
            int ax = 0;
            if (tMax[1] < tMax[ax]) ax = 1;
            if (tMax[2] < tMax[ax]) ax = 2;
            const T cap = (tMax[ax] - t_cur) * w;
            if (l_rem <= cap) {
                t_end = t_cur + l_rem / w;
                deposit(vox, Q - q_done);
                break;
            }
            l_rem = l_rem - cap;
            acc = acc + cap;
            t_cur = tMax[ax];
            uint64_t q_cum = (uint64_t)std::llrint((double)Q * (double)(acc * il));
            if (q_cum > Q) q_cum = Q;
            deposit(vox, q_cum - q_done);
            q_done = q_cum;
            tMax[ax] = tMax[ax] + tDelta[ax];
            iv[ax] += dirn[ax];
            end_visit();                                         /* the proton has left the voxel */
            if (iv[ax] < 0 || iv[ax] >= G.n[ax]) { escaped = true; break; }
            vox = (uint64_t)iv[0] + (uint64_t)G.n[0] * ((uint64_t)iv[1] + (uint64_t)G.n[1] * (uint64_t)iv[2]);
        }
        if (escaped) {
            if (!secondary) st.escaped++;
            st.q_escaped += Q - q_done;
            for (uint64_t m = k + 1; m < S.k_end; ++m) st.q_escaped += (uint64_t)std::llrint(db.dE[m] * 16777216.0f);
            if (end_state) { for (int a = 0; a < 3; ++a) { end_state[a] = FMA(t_cur, g[a], p[a]); end_state[3 + a] = g[a]; } }
            end_history();
            return;
        }
        for (int a = 0; a < 3; ++a) p[a] = FMA(t_end, g[a], p[a]);
        branch_after(k);
    }
    if (!secondary) st.stopped++;
    end_history();
    if (end_state) { for (int a = 0; a < 3; ++a) { end_state[a] = p[a]; end_state[3 + a] = g[a]; } }
}

void fill_geometry(Geometry &G, const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
                   const Knot *table, int n_knots)
{
    G.hu = hu; G.n[0] = nx; G.n[1] = ny; G.n[2] = nz; G.sp[0] = sx; G.sp[1] = sy; G.sp[2] = sz;
    material_lut(table, n_knots, G.lut_rho, G.lut_w, G.lut_f);
}

template <class T>
int run_T(const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
          const Knot *table, int n_knots, const TrackDB *db, const Beamlet *bl, uint32_t n_bl,
          uint64_t first, uint64_t n, uint64_t stride, uint64_t seed, uint32_t flags,
          uint64_t *grid, Stats *stats, Trace *tr, T *end_state, Squares *sq = nullptr, const Secondaries *sec = nullptr)
{
    Geometry *G = new Geometry;
    fill_geometry(*G, hu, nx, ny, nz, sx, sy, sz, table, n_knots);
    Stats st; std::memset(&st, 0, sizeof st);
    int rc = 0;
    for (uint64_t m = 0; m < n; ++m) {
        uint64_t i = first + m * stride;
        Start<T> S;
        rc = start_proton<T>(*G, *db, bl, n_bl, i, seed, flags, S);
        if (rc < 0) break;
        st.protons++;
        if (S.missed) { st.missed++; continue; }
        if (!sec) { transport<T>(*G, *db, S, grid, st, tr, end_state ? end_state + 6 * m : nullptr, sq); continue; }
        std::vector<Start<T>> spawn; History hist;                          /* R15 */
        transport<T>(*G, *db, S, grid, st, tr, nullptr, sq, sec, &spawn, false, &hist);
        for (size_t b = 0; b < spawn.size(); ++b) transport<T>(*G, *db, spawn[b], grid, st, tr, nullptr, sq, nullptr, nullptr, true, &hist);
        reduce_history(hist, sq);
    }
    delete G;
    if (stats) {
        stats->protons += st.protons; stats->proton_steps += st.proton_steps; stats->deposits += st.deposits;
        stats->missed += st.missed; stats->escaped += st.escaped; stats->stopped += st.stopped;
        stats->q_replayed += st.q_replayed; stats->q_escaped += st.q_escaped;
    }
    return rc;
}

}  // namespace

extern "C" {

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    Block b = philox4x32_10(ctr[0], ctr[1], ctr[2], ctr[3], key[0], key[1]);
    for (int i = 0; i < 4; ++i) out[i] = b.w[i];
}

float oracle_signed_unit(uint32_t x) { return signed_unit(x); }
double oracle_ln(double x) { return contract_ln(x); }

/* R1: three arrays of 4096 floats indexed by HU + 1024 */
void oracle_material_lut(const Knot *table, int n_knots, float *rho, float *w, float *f_theta)
{ material_lut(table, n_knots, rho, w, f_theta); }

int oracle_energy_bin(float E0, float e_min, float e_bin) { return energy_bin(E0, e_min, e_bin); }

/* R2-R6 for a list of protons; out arrays sized n (see tests/test_oracle_sampler.py) */
int oracle_sample(const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
                  const Knot *table, int n_knots, const TrackDB *db, const Beamlet *bl, uint32_t n_bl,
                  uint64_t first, uint64_t n, uint64_t stride, uint64_t seed, uint32_t flags,
                  uint32_t *beamlet, uint32_t *track, uint64_t *k0, float *p /*3n*/, float *R /*9n*/,
                  int32_t *iv /*3n*/, int32_t *missed, float *csg /*4n: c,s,gx,gy*/)
{
    Geometry *G = new Geometry;
    fill_geometry(*G, hu, nx, ny, nz, sx, sy, sz, table, n_knots);
    int rc = 0;
    for (uint64_t m = 0; m < n; ++m) {
        Start<float> S; std::memset(&S, 0, sizeof S);
        rc = start_proton<float>(*G, *db, bl, n_bl, first + m * stride, seed, flags, S);
        if (rc < 0) break;
        beamlet[m] = S.beamlet; track[m] = S.track; k0[m] = S.k0; missed[m] = S.missed;
        for (int a = 0; a < 3; ++a) { p[3 * m + a] = S.p[a]; iv[3 * m + a] = S.iv[a]; for (int j = 0; j < 3; ++j) R[9 * m + 3 * a + j] = S.R[a][j]; }
        csg[4 * m] = S.c; csg[4 * m + 1] = S.s; csg[4 * m + 2] = S.gx; csg[4 * m + 3] = S.gy;
    }
    delete G;
    return rc;
}

/* The whole path R1-R8 in the contract's f32: ADDS into grid (nx*ny*nz u64) and into *stats. */
int oracle_run(const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
               const Knot *table, int n_knots, const TrackDB *db, const Beamlet *bl, uint32_t n_bl,
               uint64_t first, uint64_t n, uint64_t stride, uint64_t seed, uint32_t flags,
               uint64_t *grid, Stats *stats)
{
    return run_T<float>(hu, nx, ny, nz, sx, sy, sz, table, n_knots, db, bl, n_bl, first, n, stride, seed, flags,
                        grid, stats, nullptr, nullptr);
}

/* R12: the path from a phase-space array: particle m is proton first_id + m (random numbers: track
 * choice and azimuth only).  ADDS into grid and *stats. */
int oracle_run_phase_space(const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
                           const Knot *table, int n_knots, const TrackDB *db, const Particle *ps, uint64_t n,
                           uint64_t first_id, uint64_t seed, uint32_t flags, uint64_t *grid, Stats *stats)
{
    Geometry *G = new Geometry;
    fill_geometry(*G, hu, nx, ny, nz, sx, sy, sz, table, n_knots);
    Stats st; std::memset(&st, 0, sizeof st);
    int rc = 0;
    for (uint64_t m = 0; m < n; ++m) {
        const Beamlet B = beamlet_of(ps[m]);
        Start<float> S; S.beamlet = 0;
        rc = start_from<float>(*G, *db, B, first_id + m, seed, flags, S);
        if (rc < 0) break;
        st.protons++;
        if (S.missed) { st.missed++; continue; }
        transport<float>(*G, *db, S, grid, st, nullptr, nullptr);
    }
    delete G;
    if (stats) {
        stats->protons += st.protons; stats->proton_steps += st.proton_steps; stats->deposits += st.deposits;
        stats->missed += st.missed; stats->escaped += st.escaped; stats->stopped += st.stopped;
        stats->q_replayed += st.q_replayed; stats->q_escaped += st.q_escaped;
    }
    return rc;
}

void oracle_frame_rule(const float d[3], float e1[3], float e2[3]) { frame_rule(d, e1, e2); }

/* oracle_run plus the sum-of-squares tallies of R10 (either may be null); all three grids are ADDED to. */
int oracle_run_sq(const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
                  const Knot *table, int n_knots, const TrackDB *db, const Beamlet *bl, uint32_t n_bl,
                  uint64_t first, uint64_t n, uint64_t stride, uint64_t seed, uint32_t flags,
                  uint64_t *grid, uint64_t *sq_by_visit, uint64_t *sq_by_history, Stats *stats)
{
    Squares sq; sq.by_visit = sq_by_visit; sq.by_history = sq_by_history;
    return run_T<float>(hu, nx, ny, nz, sx, sy, sz, table, n_knots, db, bl, n_bl, first, n, stride, seed, flags,
                        grid, stats, nullptr, nullptr, &sq);
}

/* R15: oracle_run_sq for a database whose histories have secondaries (squares grids may be null). */
int oracle_run_secondaries(const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
                           const Knot *table, int n_knots, const TrackDB *db, const uint32_t *sec_first, const uint32_t *sec_track,
                           const uint32_t *sec_step, const Beamlet *bl, uint32_t n_bl,
                           uint64_t first, uint64_t n, uint64_t stride, uint64_t seed, uint32_t flags,
                           uint64_t *grid, uint64_t *sq_by_visit, uint64_t *sq_by_history, Stats *stats)
{
    Squares sq; sq.by_visit = sq_by_visit; sq.by_history = sq_by_history;
    Secondaries sec; sec.first = sec_first; sec.track = sec_track; sec.step = sec_step;
    return run_T<float>(hu, nx, ny, nz, sx, sy, sz, table, n_knots, db, bl, n_bl, first, n, stride, seed, flags,
                        grid, stats, nullptr, nullptr, &sq, &sec);
}

/* Same rules evaluated in f64 (error bounding; brute-force and Siddon comparisons). */
int oracle_run_f64(const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
                   const Knot *table, int n_knots, const TrackDB *db, const Beamlet *bl, uint32_t n_bl,
                   uint64_t first, uint64_t n, uint64_t stride, uint64_t seed, uint32_t flags,
                   uint64_t *grid, Stats *stats, double *end_state /* 6n or null */)
{
    return run_T<double>(hu, nx, ny, nz, sx, sy, sz, table, n_knots, db, bl, n_bl, first, n, stride, seed, flags,
                         grid, stats, nullptr, end_state);
}

/* f32 run that also records every deposit (voxel, share, step number) up to cap entries. */
int oracle_run_trace(const int16_t *hu, int nx, int ny, int nz, float sx, float sy, float sz,
                     const Knot *table, int n_knots, const TrackDB *db, const Beamlet *bl, uint32_t n_bl,
                     uint64_t first, uint64_t n, uint64_t stride, uint64_t seed, uint32_t flags,
                     uint64_t *grid, Stats *stats, uint64_t *tr_voxel, uint64_t *tr_share, uint32_t *tr_step,
                     uint64_t cap, uint64_t *n_trace, float *end_state /* 6n or null */)
{
    Trace tr; tr.voxel = tr_voxel; tr.share = tr_share; tr.step = tr_step; tr.cap = cap; tr.n = 0;
    int rc = run_T<float>(hu, nx, ny, nz, sx, sy, sz, table, n_knots, db, bl, n_bl, first, n, stride, seed, flags,
                          grid, stats, &tr, end_state);
    *n_trace = tr.n;
    return rc;
}

/* R9 */
void oracle_to_gy(const uint64_t *grid, const int16_t *hu, uint64_t n_vox, float sx, float sy, float sz,
                  const Knot *table, int n_knots, float *dose)
{
    float *rho = new float[3 * N_MAT];
    material_lut(table, n_knots, rho, rho + N_MAT, rho + 2 * N_MAT);
    const double K = 1.602176634e-7 * 5.9604644775390625e-08;
    const double V = (double)sx * (double)sy * (double)sz;
    for (uint64_t v = 0; v < n_vox; ++v)
        dose[v] = (float)(((double)grid[v] * K) / ((double)rho[mat_index(hu[v])] * V));
    delete[] rho;
}

}  // extern "C"
