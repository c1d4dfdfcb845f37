// tune.cu — the launch-parameter database of the auto-tuner (section 4: "measures the execution
// time as a function of N_t and determines the best value and stores it in a database").  The measuring is
// done by paper_1212_0785_b200/autotune.py through the public calls; this file only holds the table the
// launchers consult: per (lattice extents, precision, ALL-or-parity subset, kernel) a kernel variant, a block
// shape (4-D tile for the stencil kernel) and a thread count (site-local kernels).  Host only, mutex-guarded.
#include <cstring>
#include <mutex>
#include <vector>

#include "qcd_internal.h"

namespace qcd {

namespace {
struct Entry {
    int L[4], prec, par_subset, kernel;
    TuneCfg cfg;
};
std::mutex g_mu;
std::vector<Entry> g_table;

bool same_key(const Entry &e, const LatP &p, int prec, int par_subset, int kernel) {
    return !memcmp(e.L, p.L, sizeof e.L) && e.prec == prec && e.par_subset == par_subset && e.kernel == kernel;
}
}  // namespace

bool tune_lookup(const qcd_lattice *lat, int prec, int subset, int kernel, TuneCfg &out) {
    std::lock_guard<std::mutex> g(g_mu);
    for (const Entry &e : g_table)
        if (same_key(e, lat->p, prec, subset != QCD_ALL, kernel)) {
            out = e.cfg;
            return true;
        }
    return false;
}

void tune_store(const qcd_lattice *lat, int prec, int subset, int kernel, const TuneCfg &cfg) {
    std::lock_guard<std::mutex> g(g_mu);
    for (Entry &e : g_table)
        if (same_key(e, lat->p, prec, subset != QCD_ALL, kernel)) {
            e.cfg = cfg;
            return;
        }
    Entry e;
    memcpy(e.L, lat->p.L, sizeof e.L);
    e.prec = prec;
    e.par_subset = subset != QCD_ALL;
    e.kernel = kernel;
    e.cfg = cfg;
    g_table.push_back(e);
}

void tune_clear_all() {
    std::lock_guard<std::mutex> g(g_mu);
    g_table.clear();
}

}  // namespace qcd
