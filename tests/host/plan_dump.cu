// Host-only dump of the sweep's work decomposition (csrc/em_tile.cuh) for tests/test_plan_host.py:
//   plan_dump nx ny nz sizeof_real n_sm forced_zsplit thermal  ->  one JSON object on stdout
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "../../paper_2603_07038_b200/csrc/em_tile.cuh"

int main(int argc, char **argv) {
    if (argc < 8) return 2;
    const int nx = atoi(argv[1]), ny = atoi(argv[2]), nz = atoi(argv[3]), sz = atoi(argv[4]), n_sm = atoi(argv[5]);
    const int forced = atoi(argv[6]), thermal = atoi(argv[7]);
    const em::SweepPlan f = em::make_sweep_plan(nx, ny, nz, sz, n_sm, forced, thermal != 0);
    std::vector<int> order((size_t)f.n_tiles * f.nzs);
    em::launch_order(f, order.data());
    printf("{\"V\": %d, \"TXo\": %d, \"TY\": %d, \"ntx\": %d, \"nty\": %d, \"n_tiles\": %d, \"nzs\": %d, \"kb\": [", f.V, f.TXo, f.TY, f.ntx, f.nty, f.n_tiles, f.nzs);
    for (int c = 0; c <= em::kSweepMaxZSplit; ++c) printf("%d%s", f.kb[c], c < em::kSweepMaxZSplit ? ", " : "");
    printf("], \"order\": [");
    for (size_t n = 0; n < order.size(); ++n) printf("%d%s", order[n], n + 1 < order.size() ? ", " : "");
    // the tiles that compute E' at a few nodes (owner + low-border recompute halos)
    printf("], \"tiles_of_node\": [");
    const int probes[4][2] = {{0, 0}, {f.TXo, f.TY}, {nx, ny}, {f.TXo, 1}};
    for (int q = 0; q < 4; ++q) {
        int out[4]; const int n = em::tiles_of_node(f, probes[q][0] <= nx ? probes[q][0] : nx, probes[q][1] <= ny ? probes[q][1] : ny, out);
        printf("[");
        for (int t = 0; t < n; ++t) printf("%d%s", out[t], t + 1 < n ? ", " : "");
        printf("]%s", q < 3 ? ", " : "");
    }
    printf("]}\n");
    return 0;
}
