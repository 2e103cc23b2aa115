// Host layout builder: mask V < V_cut -> active set M -> 8x8 column tiles with one
// 64-bit occupancy mask per z-plane, compact storage order, tile neighbour table, work items.
// Definitions: DESIGN.md "Layout tables".  Prior art: PAPER.md:50-58 (region of interest from the
// Thomas-Fermi density, Eq. 5), :81-85 (block post-selection and index tables).
//
// Compiled with -ffp-contract=off: the mask must be bit-exact against an independent evaluation, so the
// potential is evaluated in the fixed order of DESIGN.md R2 with one rounding per operation.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <limits>
#include <numeric>

#include "gpe_internal.h"

namespace gpe {

namespace {

struct TileTmp {
    int32_t i, j, zlo, zhi;
    std::vector<uint64_t> masks;  // [zhi - zlo]
};

inline double coord(int32_t i, int32_t n, double h, double c) {
    // x_i = ((double)i - 0.5 (n-1)) h + c : the bracket is exact (R1)
    return ((double)i - 0.5 * (double)(n - 1)) * h + c;
}

// V_mask at one point (R2 evaluation order, R13 union closed form).
// sxy = ax x^2 + ay y^2 and szz = az z^2 are passed in so the caller can hoist them; the sum
// (ax x^2 + ay y^2) + az z^2 is the left-to-right order of R2.
inline double mask_potential(const gpe_potential& p, double sxy, double szz) {
    double s = sxy + szz;
    double u = 0.5 * s;
    if (p.kind == GPE_POT_HARMONIC) return u;
    double dl;
    if (p.mask_mode == GPE_MASK_AT_DELTA0) {
        dl = p.delta0;
    } else if (p.mask_mode == GPE_MASK_AT_DELTA1) {
        dl = p.delta1;
    } else {
        double lo = std::min(p.delta0, p.delta1), hi = std::max(p.delta0, p.delta1);
        dl = std::min(std::max(u, lo), hi);
    }
    double d = u - dl;
    return std::sqrt(d * d + p.omega * p.omega) - p.omega;
}

int check_box(const gpe_box& b, std::string* err) {
    if (b.nx < 1 || b.ny < 1 || b.nz < 1) { *err = "box dimensions must be >= 1"; return GPE_ERR_INVALID_ARG; }
    if (!(b.h > 0.0) || !std::isfinite(b.h)) { *err = "h must be finite and > 0"; return GPE_ERR_INVALID_ARG; }
    if (!std::isfinite(b.hy) || !std::isfinite(b.hz)) { *err = "hy and hz must be finite (<= 0: same as h)"; return GPE_ERR_INVALID_ARG; }
    if (b.reserved != 0) { *err = "gpe_box.reserved must be 0"; return GPE_ERR_INVALID_ARG; }
    long double npts = (long double)b.nx * b.ny * b.nz;
    if (npts > 4.0e18L) { *err = "box has more than 2^62 points"; return GPE_ERR_INVALID_ARG; }
    return GPE_OK;
}

int check_pot(const gpe_potential& p, std::string* err) {
    if (p.kind != GPE_POT_HARMONIC && p.kind != GPE_POT_DRESSED) { *err = "unknown potential kind"; return GPE_ERR_INVALID_ARG; }
    if (p.mask_mode < GPE_MASK_AT_DELTA0 || p.mask_mode > GPE_MASK_UNION) { *err = "unknown mask_mode"; return GPE_ERR_INVALID_ARG; }
    return GPE_OK;
}

// Tables from the per-tile masks (tiles ascending in i*nty + j).
int finish_layout(std::vector<TileTmp>& tiles, GridHost* g, std::string* err) {
    const gpe_box& b = g->box;
    const int tx = g->tx, ty = g->ty, zt = g->zt;
    g->ntx = (b.nx + tx - 1) / tx;
    g->nty = (b.ny + ty - 1) / ty;
    const int64_t nt = (int64_t)tiles.size();
    if (nt > (int64_t)std::numeric_limits<int32_t>::max() / 8) { *err = "too many tiles"; return GPE_ERR_UNSUPPORTED; }

    g->tile_xy.resize(2 * nt);
    g->tile_zlo.resize(nt);
    g->tile_zhi.resize(nt);
    g->tile_entry_base.resize(nt);
    g->tile_nbr.assign(4 * nt, -1);

    int64_t n_slabs = 0;
    for (int64_t k = 0; k < nt; ++k) {
        g->tile_xy[2 * k] = tiles[k].i;
        g->tile_xy[2 * k + 1] = tiles[k].j;
        g->tile_zlo[k] = tiles[k].zlo;
        g->tile_zhi[k] = tiles[k].zhi;
        g->tile_entry_base[k] = n_slabs;
        n_slabs += tiles[k].zhi - tiles[k].zlo;
    }
    g->slab_mask.resize(n_slabs);
    g->slab_base.resize(n_slabs);

    // neighbour table through a dense (ntx x nty) directory of present tiles
    std::vector<int32_t> dir((size_t)g->ntx * g->nty, -1);
    for (int64_t k = 0; k < nt; ++k) dir[(size_t)tiles[k].i * g->nty + tiles[k].j] = (int32_t)k;
    static const int di[4] = {-1, 1, 0, 0}, dj[4] = {0, 0, -1, 1};
    for (int64_t k = 0; k < nt; ++k)
        for (int q = 0; q < 4; ++q) {
            int ii = tiles[k].i + di[q], jj = tiles[k].j + dj[q];
            if (ii >= 0 && ii < g->ntx && jj >= 0 && jj < g->nty) g->tile_nbr[4 * k + q] = dir[(size_t)ii * g->nty + jj];
        }

    // slab masks, storage bases, work items, per-column counts
    std::vector<int64_t> col_count((size_t)b.nx * b.ny + 1, 0);
    int64_t pos = 0;
    g->wi_tile.clear(); g->wi_z0.clear(); g->wi_nz.clear();
    for (int64_t k = 0; k < nt; ++k) {
        const TileTmp& t = tiles[k];
        const int64_t e0 = g->tile_entry_base[k];
        const int nzl = t.zhi - t.zlo;
        for (int z = 0; z < nzl; ++z) {
            uint64_t m = t.masks[z];
            g->slab_mask[e0 + z] = m;
            g->slab_base[e0 + z] = pos;
            pos += __builtin_popcountll(m);
            while (m) {
                int bit = __builtin_ctzll(m);
                m &= m - 1;
                int ix = t.i * tx + bit / ty, iy = t.j * ty + bit % ty;
                col_count[(size_t)ix * b.ny + iy + 1] += 1;
            }
        }
        // work items: maximal runs of non-empty slabs, a run of length l split into ceil(l/zt) pieces
        int z = 0;
        while (z < nzl) {
            if (t.masks[z] == 0) { ++z; continue; }
            int z1 = z;
            while (z1 < nzl && t.masks[z1] != 0) ++z1;
            const int64_t l = z1 - z;
            const int64_t kk = (l + zt - 1) / zt;
            for (int64_t i = 0; i < kk; ++i) {
                int64_t s0 = z + (i * l) / kk, s1 = z + ((i + 1) * l) / kk;
                g->wi_tile.push_back((int32_t)k);
                g->wi_z0.push_back((int32_t)(t.zlo + s0));
                g->wi_nz.push_back((int32_t)(s1 - s0));
            }
            z = z1;
        }
    }
    g->n_active = pos;

    // canonical order = ascending L = (ix*ny + iy)*nz + iz: columns ascending, z ascending in a column
    for (size_t c = 1; c < col_count.size(); ++c) col_count[c] += col_count[c - 1];  // now col_start
    g->active_idx.resize(pos);
    g->storage_to_canonical.resize(pos);
    std::vector<int64_t>& cursor = col_count;  // cursor[c] = next canonical rank of column c
    int64_t s = 0;
    for (int64_t k = 0; k < nt; ++k) {
        const TileTmp& t = tiles[k];
        const int nzl = t.zhi - t.zlo;
        for (int z = 0; z < nzl; ++z) {
            uint64_t m = t.masks[z];
            while (m) {
                int bit = __builtin_ctzll(m);
                m &= m - 1;
                int ix = t.i * tx + bit / ty, iy = t.j * ty + bit % ty;
                size_t c = (size_t)ix * b.ny + iy;
                int64_t rank = cursor[c]++;
                g->storage_to_canonical[s++] = rank;
                g->active_idx[rank] = ((int64_t)ix * b.ny + iy) * b.nz + (t.zlo + z);
            }
        }
        std::vector<uint64_t>().swap(tiles[k].masks);
    }
    return GPE_OK;
}

}  // namespace

double delta_of_t(const gpe_potential& pot, double t) {
    if (pot.t_ramp <= 0.0) return pot.delta0;
    double s = t / pot.t_ramp;
    s = std::min(std::max(s, 0.0), 1.0);
    return pot.delta0 + (pot.delta1 - pot.delta0) * s;
}

int build_layout_from_potential(const gpe_box& box, const gpe_potential& pot, double v_cut, int halo_width,
                                GridHost* g, std::string* err) {
    int rc = check_box(box, err);
    if (rc) return rc;
    rc = check_pot(pot, err);
    if (rc) return rc;
    if (halo_width < 0 || halo_width > 8) { *err = "halo_width must be in 0..8"; return GPE_ERR_INVALID_ARG; }
    if (std::isnan(v_cut)) { *err = "v_cut is NaN"; return GPE_ERR_INVALID_ARG; }
    g->box = box; g->pot = pot; g->v_cut = v_cut; g->halo_width = halo_width;
    const int tx = g->tx, ty = g->ty;
    const int ntx = (box.nx + tx - 1) / tx, nty = (box.ny + ty - 1) / ty;

    // z-dependent term computed once; one tile-row (tx x-planes) per parallel task
    std::vector<double> zz(box.nz);
    for (int iz = 0; iz < box.nz; ++iz) { double z = coord(iz, box.nz, box.hz > 0.0 ? box.hz : box.h, box.center[2]); zz[iz] = pot.az * (z * z); }

    std::vector<std::vector<TileTmp>> rows(ntx);
    std::atomic<bool> oom{false};   // set by any thread whose allocation fails (no exception may leave the region)
#pragma omp parallel
    {
        std::vector<uint64_t> buf;
        try { buf.resize((size_t)nty * box.nz); } catch (...) { oom.store(true, std::memory_order_relaxed); }
#pragma omp for schedule(dynamic, 1)
        for (int i = 0; i < ntx; ++i) {
            if (oom.load(std::memory_order_relaxed)) continue;
            try {
            std::fill(buf.begin(), buf.end(), 0ull);
            for (int lx = 0; lx < tx; ++lx) {
                int ix = i * tx + lx;
                if (ix >= box.nx) break;
                double x = coord(ix, box.nx, box.h, box.center[0]);
                for (int iy = 0; iy < box.ny; ++iy) {
                    double y = coord(iy, box.ny, box.hy > 0.0 ? box.hy : box.h, box.center[1]);
                    const double sxy = pot.ax * (x * x) + pot.ay * (y * y);
                    const int j = iy / ty;
                    const uint64_t bit = 1ull << (lx * ty + iy % ty);
                    uint64_t* mrow = &buf[(size_t)j * box.nz];
                    for (int iz = 0; iz < box.nz; ++iz)
                        if (mask_potential(pot, sxy, zz[iz]) < v_cut) mrow[iz] |= bit;
                }
            }
            for (int j = 0; j < nty; ++j) {
                const uint64_t* mrow = &buf[(size_t)j * box.nz];
                int zlo = 0, zhi = box.nz;
                while (zlo < box.nz && mrow[zlo] == 0) ++zlo;
                if (zlo == box.nz) continue;
                while (mrow[zhi - 1] == 0) --zhi;
                TileTmp t;
                t.i = i; t.j = j; t.zlo = zlo; t.zhi = zhi;
                t.masks.assign(mrow + zlo, mrow + zhi);
                rows[i].push_back(std::move(t));
            }
            } catch (...) { oom.store(true, std::memory_order_relaxed); }
        }
    }
    if (oom.load()) { *err = "out of host memory in the layout builder"; return GPE_ERR_OUT_OF_MEMORY; }
    std::vector<TileTmp> tiles;
    for (int i = 0; i < ntx; ++i)
        for (auto& t : rows[i]) tiles.push_back(std::move(t));
    rows.clear();
    try {
        return finish_layout(tiles, g, err);
    } catch (const std::bad_alloc&) {
        *err = "out of host memory in the layout builder";
        return GPE_ERR_OUT_OF_MEMORY;
    }
}

int build_layout_from_indices(const gpe_box& box, const gpe_potential& pot, const int64_t* active, int64_t n,
                              int halo_width, GridHost* g, std::string* err) {
    int rc = check_box(box, err);
    if (rc) return rc;
    rc = check_pot(pot, err);
    if (rc) return rc;
    if (halo_width < 0 || halo_width > 8) { *err = "halo_width must be in 0..8"; return GPE_ERR_INVALID_ARG; }
    if (n < 0 || (n > 0 && !active)) { *err = "bad active index list"; return GPE_ERR_INVALID_ARG; }
    const int64_t npts = (int64_t)box.nx * box.ny * box.nz;
    for (int64_t k = 0; k < n; ++k) {
        if (active[k] < 0 || active[k] >= npts) { *err = "active index outside the box"; return GPE_ERR_INVALID_ARG; }
        if (k && active[k] <= active[k - 1]) { *err = "active indices must be strictly ascending"; return GPE_ERR_INVALID_ARG; }
    }
    g->box = box; g->pot = pot; g->v_cut = std::numeric_limits<double>::quiet_NaN(); g->halo_width = halo_width;
    const int tx = g->tx, ty = g->ty;
    const int nty = (box.ny + ty - 1) / ty;
    try {
        // sort point ranks by (tile, z); bits are OR-ed so their order does not matter
        std::vector<int64_t> tid(n);
        for (int64_t k = 0; k < n; ++k) {
            int64_t L = active[k];
            int64_t ix = L / ((int64_t)box.ny * box.nz), iy = (L / box.nz) % box.ny;
            tid[k] = (ix / tx) * nty + (iy / ty);
        }
        std::vector<int64_t> ord(n);
        std::iota(ord.begin(), ord.end(), (int64_t)0);
        std::stable_sort(ord.begin(), ord.end(), [&](int64_t a, int64_t b) { return tid[a] < tid[b]; });
        std::vector<TileTmp> tiles;
        int64_t a = 0;
        while (a < n) {
            int64_t e = a;
            int zlo = box.nz, zhi = 0;
            while (e < n && tid[ord[e]] == tid[ord[a]]) {
                int iz = (int)(active[ord[e]] % box.nz);
                zlo = std::min(zlo, iz); zhi = std::max(zhi, iz + 1);
                ++e;
            }
            TileTmp t;
            t.i = (int32_t)(tid[ord[a]] / nty); t.j = (int32_t)(tid[ord[a]] % nty); t.zlo = zlo; t.zhi = zhi;
            t.masks.assign(zhi - zlo, 0ull);
            for (int64_t q = a; q < e; ++q) {
                int64_t L = active[ord[q]];
                int64_t ix = L / ((int64_t)box.ny * box.nz), iy = (L / box.nz) % box.ny, iz = L % box.nz;
                t.masks[iz - zlo] |= 1ull << ((ix % tx) * ty + (iy % ty));
            }
            tiles.push_back(std::move(t));
            a = e;
        }
        return finish_layout(tiles, g, err);
    } catch (const std::bad_alloc&) {
        *err = "out of host memory in the layout builder";
        return GPE_ERR_OUT_OF_MEMORY;
    }
}

// S = M u star-halo(M, halo_width) clipped to the box (R3, R4), ascending L.
void build_stored_indices(GridHost* g) {
    if (g->stored_ready) return;
    const gpe_box& b = g->box;
    const int64_t strides[3] = {(int64_t)b.ny * b.nz, b.nz, 1};
    const int64_t dims[3] = {b.nx, b.ny, b.nz};
    std::vector<int64_t> all(g->active_idx);
    for (int64_t k = 0; k < g->n_active; ++k) {
        int64_t L = g->active_idx[k];
        int64_t c[3] = {L / strides[0], (L / b.nz) % b.ny, L % b.nz};
        for (int axis = 0; axis < 3; ++axis)
            for (int s = -g->halo_width; s <= g->halo_width; ++s) {
                if (s == 0) continue;
                int64_t q = c[axis] + s;
                if (q >= 0 && q < dims[axis]) all.push_back(L + s * strides[axis]);
            }
    }
    std::sort(all.begin(), all.end());
    all.erase(std::unique(all.begin(), all.end()), all.end());
    g->stored_idx.swap(all);
    g->stored_ready = true;
}

}  // namespace gpe
