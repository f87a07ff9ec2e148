/*
 * oracle/ccl_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU statement of what the hot path of
 * Komura, "A generalized GPU-based connected component labeling algorithm"
 * (arXiv 1603.08357; /root/reference/PAPER.md) computes, plus the CPU side of
 * the seeded workload generators.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this file.  It
 * shares no code, header, table or helper with the CUDA library in
 * paper_1603_08357_b200/csrc/, and neither includes the other.
 *
 * What is pinned by what (tests/test_oracle_*.py, all `-m "not gpu"`):
 *   oracle_label / oracle_label_bits   Fig. 1 -> Fig. 4 worked example, BFS brute force,
 *                                      closed forms (p=0, p=1, paths), invariants, p_c crossings
 *   oracle_stats                       brute-force counting in the tests, sum rule
 *   oracle_wrap                        BFS on the unwrapped cover (tiny lattices), straight-row cases
 *   oracle_philox4x32_10               published known-answer vectors (Salmon et al., SC'11 test suite)
 *   oracle_gen_*                       degree / count / simplicity properties, nestedness
 * No function here is "parity unpinned".
 *
 * Readings of the paper adopted here are listed in DESIGN.md ("Readings").
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------------
 * 1. Labeling.  Definition ("The label of each cluster depends on the minimum site
 *    number in each cluster"): labels[i] = min{ j : j connected to i through occupied bonds }.
 *    Computed as BASELINE.json:north_star prescribes: weighted union-find with path compression,
 *    then one ascending sweep that names every component after the first (= smallest) site
 *    that reaches its root.
 * ---------------------------------------------------------------------------------------------- */

static int32_t uf_find(int32_t *parent, int32_t x)
{
    int32_t r = x;
    while (parent[r] != r) r = parent[r];
    while (parent[x] != r) {            /* path compression */
        int32_t nx = parent[x];
        parent[x] = r;
        x = nx;
    }
    return r;
}

static void uf_union(int32_t *parent, int32_t *size, int32_t a, int32_t b)
{
    int32_t ra = uf_find(parent, a);
    int32_t rb = uf_find(parent, b);
    if (ra == rb) return;
    if (size[ra] < size[rb]) { int32_t t = ra; ra = rb; rb = t; }   /* smaller tree under larger; tie: second under first */
    parent[rb] = ra;
    size[ra] += size[rb];
}

/* occ_kind: 0 = all bonds occupied (occ ignored), 1 = uint8 per bond, 2 = bit b&31 of uint32 word b>>5 */
static int label_impl(int64_t n_sites, int64_t n_bonds, const int32_t *src, const int32_t *dst,
                      const void *occ, int occ_kind, int32_t *labels)
{
    if (n_sites < 0 || n_bonds < 0 || n_sites > 2147483647LL) return 1;
    if (n_sites == 0) return 0;
    int32_t *parent = (int32_t *)malloc((size_t)n_sites * sizeof(int32_t));
    int32_t *size   = (int32_t *)malloc((size_t)n_sites * sizeof(int32_t));
    if (!parent || !size) { free(parent); free(size); return 2; }
    for (int64_t i = 0; i < n_sites; ++i) { parent[i] = (int32_t)i; size[i] = 1; }

    const uint8_t  *occ8  = (const uint8_t *)occ;
    const uint32_t *occ32 = (const uint32_t *)occ;
    for (int64_t b = 0; b < n_bonds; ++b) {
        int on = 1;
        if (occ_kind == 1) on = occ8[b] != 0;
        else if (occ_kind == 2) on = (occ32[b >> 5] >> (b & 31)) & 1u;
        if (!on) continue;
        int32_t u = src[b], v = dst[b];
        if (u < 0 || v < 0 || u >= n_sites || v >= n_sites) { free(parent); free(size); return 3; }
        uf_union(parent, size, u, v);
    }

    /* canonical form: ascending sweep; the first site that reaches a root is that component's minimum */
    int32_t *minidx = size;                       /* reuse: size[] is not needed any more */
    for (int64_t i = 0; i < n_sites; ++i) minidx[i] = -1;
    for (int64_t i = 0; i < n_sites; ++i) {
        int32_t r = uf_find(parent, (int32_t)i);
        if (minidx[r] < 0) minidx[r] = (int32_t)i;
        labels[i] = minidx[r];
    }
    free(parent); free(size);
    return 0;
}

int oracle_label(int64_t n_sites, int64_t n_bonds, const int32_t *src, const int32_t *dst,
                 const uint8_t *occupied, int32_t *labels)
{
    return label_impl(n_sites, n_bonds, src, dst, occupied, occupied ? 1 : 0, labels);
}

int oracle_label_bits(int64_t n_sites, int64_t n_bonds, const int32_t *src, const int32_t *dst,
                      const uint32_t *occupied_bits, int32_t *labels)
{
    return label_impl(n_sites, n_bonds, src, dst, occupied_bits, occupied_bits ? 2 : 0, labels);
}

/* ------------------------------------------------------------------------------------------------
 * 2. Cluster statistics from canonical labels (reading R8; the paper itself measures only
 *    R_span).  size[l] = #{i : labels[i] == l}.
 * ---------------------------------------------------------------------------------------------- */
typedef struct {
    int64_t  n_clusters;      /* #{i : labels[i] == i}                                   */
    int64_t  largest;         /* max cluster size                                        */
    int64_t  largest_label;   /* label of that cluster; ties -> smallest label           */
    uint64_t sum_s2;          /* sum over clusters of size^2                             */
} oracle_stats_t;

int oracle_stats(int64_t n_sites, const int32_t *labels, oracle_stats_t *out,
                 int64_t *hist_dense, int32_t n_dense, int64_t *hist_log2 /* 32 entries */)
{
    if (n_sites < 0) return 1;
    int64_t *size = (int64_t *)calloc((size_t)(n_sites > 0 ? n_sites : 1), sizeof(int64_t));
    if (!size) return 2;
    for (int64_t i = 0; i < n_sites; ++i) {
        if (labels[i] < 0 || labels[i] >= n_sites) { free(size); return 3; }
        size[labels[i]] += 1;
    }
    out->n_clusters = 0; out->largest = 0; out->largest_label = -1; out->sum_s2 = 0;
    if (hist_dense) for (int32_t s = 0; s <= n_dense; ++s) hist_dense[s] = 0;   /* n_dense+1 entries, [0] unused */
    if (hist_log2)  for (int k = 0; k < 32; ++k) hist_log2[k] = 0;
    for (int64_t l = 0; l < n_sites; ++l) {
        int64_t s = size[l];
        if (s == 0) continue;
        out->n_clusters += 1;
        out->sum_s2 += (uint64_t)s * (uint64_t)s;
        if (s > out->largest) { out->largest = s; out->largest_label = l; }
        if (hist_dense && s <= n_dense) hist_dense[s] += 1;
        if (hist_log2) { int k = 0; while ((s >> (k + 1)) != 0) ++k; hist_log2[k] += 1; }
    }
    free(size);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * 3. Wrapping on a periodic lattice (reading R7 of "spanning").
 *    Every bond carries the displacement (dx,dy), in lattice cells, from src to dst on the
 *    infinite (unwrapped) lattice.  Union-find in which every site stores its displacement to its
 *    parent; an occupied bond whose two ends already share a root closes a cycle, and the cycle's
 *    winding vector is the mismatch between the stored displacements and the bond's own.
 *    out[0] = some cluster has a cycle with non-zero x-winding, out[1] = same for y.
 * ---------------------------------------------------------------------------------------------- */
static int32_t wfind(int32_t *parent, int32_t *px, int32_t *py, int32_t x, int32_t *ox, int32_t *oy)
{
    /* returns root of x and (ox,oy) = position(x) - position(root), without compression (plain and slow) */
    int32_t sx = 0, sy = 0;
    while (parent[x] != x) { sx += px[x]; sy += py[x]; x = parent[x]; }
    *ox = sx; *oy = sy;
    return x;
}

int oracle_wrap(int64_t n_sites, int64_t n_bonds, const int32_t *src, const int32_t *dst,
                const int8_t *dx, const int8_t *dy, const uint8_t *occupied, int32_t out[2])
{
    if (n_sites < 0 || n_bonds < 0) return 1;
    int32_t *parent = (int32_t *)malloc((size_t)(n_sites + 1) * sizeof(int32_t));
    int32_t *px = (int32_t *)calloc((size_t)(n_sites + 1), sizeof(int32_t));   /* position(x) - position(parent[x]) */
    int32_t *py = (int32_t *)calloc((size_t)(n_sites + 1), sizeof(int32_t));
    int32_t *size = (int32_t *)malloc((size_t)(n_sites + 1) * sizeof(int32_t));
    if (!parent || !px || !py || !size) { free(parent); free(px); free(py); free(size); return 2; }
    for (int64_t i = 0; i < n_sites; ++i) { parent[i] = (int32_t)i; size[i] = 1; }
    out[0] = 0; out[1] = 0;
    for (int64_t b = 0; b < n_bonds; ++b) {
        if (occupied && !occupied[b]) continue;
        int32_t u = src[b], v = dst[b];
        int32_t ux, uy, vx, vy;
        int32_t ru = wfind(parent, px, py, u, &ux, &uy);
        int32_t rv = wfind(parent, px, py, v, &vx, &vy);
        /* the bond says position(v) = position(u) + (dx,dy) */
        if (ru == rv) {
            int32_t mx = (ux + dx[b]) - vx;     /* winding of the cycle closed by this bond, times L */
            int32_t my = (uy + dy[b]) - vy;
            if (mx != 0) out[0] = 1;
            if (my != 0) out[1] = 1;
        } else if (size[ru] >= size[rv]) {
            /* hang rv under ru: position(rv) - position(ru) = position(u)+d-vx' ... */
            parent[rv] = ru;
            px[rv] = ux + dx[b] - vx;
            py[rv] = uy + dy[b] - vy;
            size[ru] += size[rv];
        } else {
            parent[ru] = rv;
            px[ru] = vx - dx[b] - ux;
            py[ru] = vy - dy[b] - uy;
            size[rv] += size[ru];
        }
    }
    free(parent); free(px); free(py); free(size);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * 4. Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11).
 *    BASELINE.json asks for seeded Philox masks; the paper used cuRAND XORWOW and prints
 *    no per-seed output, so nothing depends on matching its stream (reading R10).
 * ---------------------------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------------------------------------
 * 5. Workload generators (the paper names the lattices only).
 * ---------------------------------------------------------------------------------------------- */

/* Triangular lattice, L x L periodic: site s = y*L + x; bond 3s+k joins s to (x+1,y), (x,y+1), (x+1,y+1). */
int oracle_gen_triangular(int32_t L, int32_t *src, int32_t *dst, int8_t *dx, int8_t *dy)
{
    if (L < 1) return 1;
    static const int ddx[3] = {1, 0, 1}, ddy[3] = {0, 1, 1};
    for (int64_t y = 0; y < L; ++y)
        for (int64_t x = 0; x < L; ++x) {
            int64_t s = y * L + x;
            for (int k = 0; k < 3; ++k) {
                int64_t xx = (x + ddx[k]) % L, yy = (y + ddy[k]) % L;
                src[3 * s + k] = (int32_t)s;
                dst[3 * s + k] = (int32_t)(yy * L + xx);
                if (dx) dx[3 * s + k] = (int8_t)ddx[k];
                if (dy) dy[3 * s + k] = (int8_t)ddy[k];
            }
        }
    return 0;
}

/* Honeycomb lattice as L x L periodic two-site cells: cell c = y*L + x, A = 2c, B = 2c+1;
 * bond 3c+0 = A(c)-B(c), 3c+1 = B(c)-A(x+1,y), 3c+2 = B(c)-A(x,y+1).  Displacements count cell translations. */
int oracle_gen_honeycomb(int32_t L, int32_t *src, int32_t *dst, int8_t *dx, int8_t *dy)
{
    if (L < 1) return 1;
    for (int64_t y = 0; y < L; ++y)
        for (int64_t x = 0; x < L; ++x) {
            int64_t c = y * L + x;
            int64_t cr = y * L + (x + 1) % L;
            int64_t cu = ((y + 1) % L) * L + x;
            src[3 * c + 0] = (int32_t)(2 * c);     dst[3 * c + 0] = (int32_t)(2 * c + 1);
            src[3 * c + 1] = (int32_t)(2 * c + 1); dst[3 * c + 1] = (int32_t)(2 * cr);
            src[3 * c + 2] = (int32_t)(2 * c + 1); dst[3 * c + 2] = (int32_t)(2 * cu);
            if (dx) { dx[3 * c + 0] = 0; dx[3 * c + 1] = 1; dx[3 * c + 2] = 0; }
            if (dy) { dy[3 * c + 0] = 0; dy[3 * c + 1] = 0; dy[3 * c + 2] = 1; }
        }
    return 0;
}

/* Bernoulli(p) occupancy: T = floor(p * 2^32); bond b occupied <=> word (b&3) of
 * Philox4x32-10(counter = (b>>2 lo, b>>2 hi, realization, 0), key = (seed lo, seed hi)) < T; p >= 1 -> all. */
int oracle_gen_occupancy(int64_t n_bonds, double p, uint64_t seed, uint32_t realization,
                         uint8_t *mask_or_null, uint32_t *bits_or_null)
{
    if (n_bonds < 0 || !(p >= 0.0)) return 1;
    int all = (p >= 1.0);
    uint32_t T = all ? 0u : (uint32_t)(p * 4294967296.0);
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    if (bits_or_null) memset(bits_or_null, 0, (size_t)((n_bonds + 31) / 32) * sizeof(uint32_t));
    for (int64_t q = 0; 4 * q < n_bonds; ++q) {
        uint32_t ctr[4] = { (uint32_t)q, (uint32_t)((uint64_t)q >> 32), realization, 0u };
        uint32_t w[4];
        oracle_philox4x32_10(ctr, key, w);
        for (int j = 0; j < 4; ++j) {
            int64_t b = 4 * q + j;
            if (b >= n_bonds) break;
            int on = all || (w[j] < T);
            if (mask_or_null) mask_or_null[b] = (uint8_t)on;
            if (bits_or_null && on) bits_or_null[b >> 5] |= (1u << (b & 31));
        }
    }
    return 0;
}

/* ---- random z-regular graph by the configuration model ("Bethe substitute", BASELINE.json configs 4, 5) ---- */

typedef struct { uint64_t key; uint32_t val; } kv_t;

/* stable LSD radix sort of (key, val) by key, 8 bits per pass; val order is preserved among equal keys */
static int radix_sort_kv(kv_t *a, int64_t n)
{
    kv_t *tmp = (kv_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(kv_t));
    if (!tmp) return 1;
    kv_t *in = a, *out = tmp;
    for (int pass = 0; pass < 8; ++pass) {
        int64_t count[257];
        memset(count, 0, sizeof(count));
        int shift = 8 * pass;
        for (int64_t i = 0; i < n; ++i) count[((in[i].key >> shift) & 0xFF) + 1]++;
        for (int d = 0; d < 256; ++d) count[d + 1] += count[d];
        for (int64_t i = 0; i < n; ++i) out[count[(in[i].key >> shift) & 0xFF]++] = in[i];
        kv_t *t = in; in = out; out = t;
    }
    /* 8 passes: result is back in a */
    free(tmp);
    return 0;
}

static uint64_t pair_key(int32_t u, int32_t v)
{
    uint32_t lo = (uint32_t)(u < v ? u : v), hi = (uint32_t)(u < v ? v : u);
    return ((uint64_t)lo << 32) | hi;
}

/* how many bonds of the CURRENT graph have unordered pair key `pk`: count in the sorted snapshot of the
 * initial graph, minus removals, plus additions made by earlier repairs */
static int64_t count_sorted(const uint64_t *sorted, int64_t n, uint64_t pk)
{
    int64_t lo = 0, hi = n;
    while (lo < hi) { int64_t mid = (lo + hi) / 2; if (sorted[mid] < pk) lo = mid + 1; else hi = mid; }
    int64_t c = 0;
    while (lo + c < n && sorted[lo + c] == pk) ++c;
    return c;
}

typedef struct { uint64_t *removed; uint64_t *added; int64_t n_removed, n_added, cap; } overlay_t;

static int overlay_push(overlay_t *o, uint64_t removed, uint64_t added)
{
    if (o->n_removed >= o->cap || o->n_added >= o->cap) {
        int64_t nc = o->cap ? 2 * o->cap : 64;
        o->removed = (uint64_t *)realloc(o->removed, (size_t)nc * sizeof(uint64_t));
        o->added   = (uint64_t *)realloc(o->added,   (size_t)nc * sizeof(uint64_t));
        if (!o->removed || !o->added) return 1;
        o->cap = nc;
    }
    o->removed[o->n_removed++] = removed;
    o->added[o->n_added++] = added;
    return 0;
}

static int64_t multiplicity(const uint64_t *sorted, int64_t n, const overlay_t *o, uint64_t pk)
{
    int64_t c = count_sorted(sorted, n, pk);
    for (int64_t i = 0; i < o->n_removed; ++i) if (o->removed[i] == pk) --c;
    for (int64_t i = 0; i < o->n_added; ++i)   if (o->added[i] == pk) ++c;
    return c;
}

/* stub t (0 <= t < z*N) belongs to site t / z; key[t] = w0<<32 | w1 of Philox(counter = (t lo, t hi, 0, 1));
 * stable sort of the stubs by key; bond k joins the sites of sorted stubs 2k and 2k+1.  Defects (a self-loop,
 * or any repeat of an unordered pair after its first occurrence in bond order) are then repaired in ascending k
 * by swapping endpoints with a Philox-chosen partner bond m:  (u_k,v_k),(u_m,v_m) -> (u_k,u_m),(v_k,v_m),
 * accepted if both new bonds are non-loops, differ from each other and are absent from the graph.
 * n_repaired (optional) receives the number of defects repaired. */
int oracle_gen_regular(int64_t n_sites, int32_t z, uint64_t seed, int32_t *src, int32_t *dst, int64_t *n_repaired)
{
    if (n_sites < 1 || z < 1 || ((n_sites * z) & 1)) return 1;
    int64_t n_stubs = n_sites * z, M = n_stubs / 2;
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    kv_t *stubs = (kv_t *)malloc((size_t)n_stubs * sizeof(kv_t));
    if (!stubs) return 2;
    for (int64_t t = 0; t < n_stubs; ++t) {
        uint32_t ctr[4] = { (uint32_t)t, (uint32_t)((uint64_t)t >> 32), 0u, 1u };
        uint32_t w[4];
        oracle_philox4x32_10(ctr, key, w);
        stubs[t].key = ((uint64_t)w[0] << 32) | w[1];
        stubs[t].val = (uint32_t)t;
    }
    if (radix_sort_kv(stubs, n_stubs)) { free(stubs); return 2; }
    for (int64_t k = 0; k < M; ++k) {
        src[k] = (int32_t)(stubs[2 * k].val / (uint32_t)z);
        dst[k] = (int32_t)(stubs[2 * k + 1].val / (uint32_t)z);
    }
    free(stubs);

    /* find defects: sort (pair key, bond index); within a run of equal keys every bond but the first is a defect */
    kv_t *pk = (kv_t *)malloc((size_t)M * sizeof(kv_t));
    uint64_t *sorted = (uint64_t *)malloc((size_t)M * sizeof(uint64_t));
    uint8_t *defect = (uint8_t *)calloc((size_t)M, 1);
    if (!pk || !sorted || !defect) { free(pk); free(sorted); free(defect); return 2; }
    for (int64_t k = 0; k < M; ++k) { pk[k].key = pair_key(src[k], dst[k]); pk[k].val = (uint32_t)k; }
    if (radix_sort_kv(pk, M)) { free(pk); free(sorted); free(defect); return 2; }
    for (int64_t i = 0; i < M; ++i) {
        sorted[i] = pk[i].key;
        if (i > 0 && pk[i].key == pk[i - 1].key) defect[pk[i].val] = 1;     /* stable sort: val ascending within a run */
    }
    free(pk);
    for (int64_t k = 0; k < M; ++k) if (src[k] == dst[k]) defect[k] = 1;

    overlay_t ov; memset(&ov, 0, sizeof(ov));
    int64_t repaired = 0;
    int rc = 0;
    for (int64_t k = 0; k < M && !rc; ++k) {
        if (!defect[k]) continue;
        /* a defect flagged on the initial graph may have been cured by an earlier swap that used k as partner */
        uint64_t cur = pair_key(src[k], dst[k]);
        if (src[k] != dst[k] && multiplicity(sorted, M, &ov, cur) <= 1) continue;
        for (uint32_t attempt = 0; ; ++attempt) {
            uint32_t ctr[4] = { (uint32_t)k, (uint32_t)((uint64_t)k >> 32), attempt, 2u };
            uint32_t w[4];
            oracle_philox4x32_10(ctr, key, w);
            int64_t m = (int64_t)((((uint64_t)w[0] << 32) | w[1]) % (uint64_t)M);
            if (m == k) continue;
            int32_t uk = src[k], vk = dst[k], um = src[m], vm = dst[m];
            if (uk == um || vk == vm) continue;                       /* would create a self-loop */
            uint64_t a = pair_key(uk, um), b = pair_key(vk, vm);
            if (a == b) continue;                                     /* would create a double bond */
            if (multiplicity(sorted, M, &ov, a) != 0) continue;
            if (multiplicity(sorted, M, &ov, b) != 0) continue;
            if (overlay_push(&ov, pair_key(uk, vk), a) || overlay_push(&ov, pair_key(um, vm), b)) { rc = 2; break; }
            src[k] = uk; dst[k] = um;
            src[m] = vk; dst[m] = vm;
            ++repaired;
            break;
        }
    }
    if (n_repaired) *n_repaired = repaired;
    free(ov.removed); free(ov.added); free(sorted); free(defect);
    return rc;
}

/* Cayley tree ("Bethe lattice" of PAPER.md:189-193) with coordination number 3 and g generations in the standard
 * numbering from the centre: site 0 has children 1,2,3; site i >= 1 has children 2i+2, 2i+3.  N = 3*2^g - 2 sites,
 * N-1 bonds; bond (i-1) joins site i to its parent.  perm (optional, a permutation of 0..N-1) renumbers the sites
 * ("random position"). */
int oracle_gen_cayley3(int32_t g, const int32_t *perm_or_null, int32_t *src, int32_t *dst)
{
    if (g < 1 || g > 28) return 1;
    int64_t N = 3 * ((int64_t)1 << g) - 2;
    for (int64_t i = 1; i < N; ++i) {
        int64_t parent = (i <= 3) ? 0 : (i - 2) / 2;
        int32_t a = (int32_t)parent, b = (int32_t)i;
        if (perm_or_null) { a = perm_or_null[parent]; b = perm_or_null[i]; }
        src[i - 1] = a; dst[i - 1] = b;
    }
    return 0;
}
