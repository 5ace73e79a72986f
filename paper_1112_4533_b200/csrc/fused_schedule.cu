// fused_schedule.cu — host side of the fused multi-sub-step launches (fused_schedule.h): the geometry of cells and
// tiles, and the ticket table that says which tile of which stage a block with ticket k works on.
//
// The table is built by simulating the tickets in order. Stage 0 hands out its tiles in the traversal order of the
// plain kernel (z-chunk, t, z: DESIGN.md "Traversal order"). A cell of a later stage becomes ELIGIBLE at ticket k
// once every cell it conflicts with (fused_dep, the same enumeration the kernel waits on) has had ALL its tiles
// handed to tickets <= k - margin; each stage takes the first eligible cell in traversal order whenever it runs
// dry and gives one tile of it to every following ticket. Cells whose conflicts wrap around the lattice (first
// time slice, chunk-boundary z-planes) simply become eligible late and are picked up then. Properties (checked
// exhaustively by tests/test_fused_schedule.py on small lattices through su_fused_schedule_debug):
//   * every tile of every stage appears exactly once;
//   * every dependency of a work item of ticket k was handed to a ticket < k (no deadlock: the unfinished block
//     with the lowest ticket never waits on an unfinished block);
//   * every link-level conflict between two sub-steps is covered by a dependency.
#include <algorithm>
#include <climits>
#include <vector>

#include "su_internal.h"

namespace sug {

FusedGeom fused_make_geom(int Lx, int Ly, int Lz, int Lt, int spb, int g, int sub0, int U_force) {
    FusedGeom fg{};
    fg.Lz = Lz; fg.Lt = Lt; fg.spb = spb; fg.g = g; fg.sub0 = sub0;
    fg.plane_sites = (Lx / 2) * Ly;
    // planes per cell: the smallest divisor of Lz whose cell wastes <= 1/8 of its last tile (else the least waste)
    int best = Lz; double best_waste = 1e9;
    for (int U = 1; U <= Lz; ++U) {
        if (Lz % U) continue;
        const int sites = fg.plane_sites * U, nT = (sites + spb - 1) / spb;
        const double waste = (double)(nT * spb - sites) / sites;
        if (waste <= 0.125) { best = U; break; }
        if (waste < best_waste - 1e-12) { best_waste = waste; best = U; }
    }
    fg.U = (U_force > 0 && Lz % U_force == 0) ? U_force : best;
    fg.nzu = Lz / fg.U;
    fg.cell_sites = fg.plane_sites * fg.U;
    fg.nT = (fg.cell_sites + spb - 1) / spb;
    return fg;
}

// Returns false if the simulation does not terminate (cannot happen: stage 0 has no dependencies and every later
// stage only depends on earlier ones; guarded anyway).
bool fused_build_schedule(const FusedGeom& fg, int chunk_units, int margin, std::vector<uint32_t>& work, int& n_tickets) {
    const int g = fg.g, ncells = fg.Lt * fg.nzu, nT = fg.nT;
    if (chunk_units < 1 || chunk_units > fg.nzu) chunk_units = fg.nzu;
    while (fg.nzu % chunk_units) --chunk_units;
    if (margin < 1) margin = 1;
    // traversal order of the cells: (z-chunk, t, z within chunk)
    std::vector<int> order;
    order.reserve(ncells);
    for (int c0 = 0; c0 < fg.nzu; c0 += chunk_units)
        for (int t = 0; t < fg.Lt; ++t)
            for (int zu = c0; zu < c0 + chunk_units; ++zu) order.push_back(t * fg.nzu + zu);
    // conflicts of every (stage, cell): union over its tiles, as counter indices (a * ncells + cell')
    std::vector<std::vector<int>> deps((size_t)g * ncells);
    for (int s = 1; s < g; ++s)
        for (int c = 0; c < ncells; ++c) {
            std::vector<int>& d = deps[(size_t)s * ncells + c];
            for (int tile = 0; tile < nT; ++tile)
                for (int k = 0; k < s * FUSED_DEPS_PER_STAGE; ++k) {
                    const int idx = fused_dep(fg, s, c, tile, k);
                    if (idx >= 0) d.push_back(idx);
                }
            std::sort(d.begin(), d.end());
            d.erase(std::unique(d.begin(), d.end()), d.end());
        }
    std::vector<int> last_ticket((size_t)g * ncells, INT_MAX);     // ticket of the last tile of (stage, cell)
    std::vector<std::vector<int>> pending(g, order);                // cells not yet started, traversal order
    std::vector<int> cur_cell(g, -1), cur_tile(g, 0);
    work.clear();
    size_t remaining = (size_t)g * ncells * nT;
    int k = 0;
    const int k_limit = (ncells * nT + 1) * (g + 1) + margin * g * 4 + 16;
    for (; remaining > 0; ++k) {
        if (k > k_limit) return false;
        work.resize((size_t)(k + 1) * g, FUSED_NONE);
        for (int s = 0; s < g; ++s) {
            if (cur_cell[s] < 0) {
                std::vector<int>& pend = pending[s];
                for (size_t i = 0; i < pend.size(); ++i) {
                    bool ok = true;
                    for (int idx : deps[(size_t)s * ncells + pend[i]])
                        if (last_ticket[idx] == INT_MAX || last_ticket[idx] > k - margin) { ok = false; break; }
                    if (ok) { cur_cell[s] = pend[i]; cur_tile[s] = 0; pend.erase(pend.begin() + i); break; }
                }
            }
            if (cur_cell[s] >= 0) {
                work[(size_t)k * g + s] = (uint32_t)(cur_cell[s] * nT + cur_tile[s]);
                --remaining;
                if (++cur_tile[s] == nT) { last_ticket[(size_t)s * ncells + cur_cell[s]] = k; cur_cell[s] = -1; }
            }
        }
    }
    n_tickets = k;
    return true;
}

}  // namespace sug

// Host-only debug view of the schedule, for the CPU test of its properties (no device needed).
extern "C" su_status su_fused_schedule_debug(int Lx, int Ly, int Lz, int Lt, int sites_per_block, int n_fused, int first_substep,
                                             int planes_per_cell, int chunk_planes, int margin, uint32_t* work, size_t work_capacity,
                                             int* n_tickets, int* geom /* U, nzu, nT, cell_sites, plane_sites */) {
    using namespace sug;
    if (!n_tickets || !geom || Lx < 2 || Ly < 2 || Lz < 2 || Lt < 2 || ((Lx | Ly | Lz | Lt) & 1) || sites_per_block < 1 ||
        n_fused < 1 || n_fused > FUSED_MAX_G || first_substep < 0 || first_substep + n_fused > 8)
        return SU_EINVAL;
    const FusedGeom fg = fused_make_geom(Lx, Ly, Lz, Lt, sites_per_block, n_fused, first_substep, planes_per_cell);
    std::vector<uint32_t> w;
    int nt = 0;
    if (!fused_build_schedule(fg, chunk_planes > 0 ? std::max(1, chunk_planes / fg.U) : fg.nzu, margin, w, nt)) return SU_ESTATE;
    *n_tickets = nt;
    geom[0] = fg.U; geom[1] = fg.nzu; geom[2] = fg.nT; geom[3] = fg.cell_sites; geom[4] = fg.plane_sites;
    if (work) {
        if (work_capacity < w.size()) return SU_ENOMEM;
        std::copy(w.begin(), w.end(), work);
    }
    return SU_OK;
}

extern "C" int su_fused_dep_debug(int Lx, int Ly, int Lz, int Lt, int sites_per_block, int n_fused, int first_substep,
                                  int planes_per_cell, int stage, int cell, int tile, int k) {
    using namespace sug;
    const FusedGeom fg = fused_make_geom(Lx, Ly, Lz, Lt, sites_per_block, n_fused, first_substep, planes_per_cell);
    return fused_dep(fg, stage, cell, tile, k);
}
