// Host DAG compiler under AddressSanitizer / UndefinedBehaviorSanitizer (tests/test_abi_and_compiler.py builds and runs
// this): every mode (uniform, SB-CoS, uniform with shift; square and honeycomb; single output, all subsets, partial
// readout sets) for n = 1..8.
#include "../paper_2507_12349_b200/csrc/cos_compile.h"
#include <cstdio>
using namespace cosb;
int main()
{
    double sig[4] = {0.2, 0.0, -0.2, 0.1};
    unsigned long long total = 0;
    for (int n = 1; n <= 8; ++n)
        for (int nsub = 1; nsub <= 2; ++nsub)
            for (int mode = 0; mode < 3; ++mode)           // 0 uniform, 1 SB, 2 uniform + shift
                for (int all = 0; all < 2; ++all)
                    for (int nf = 2; nf <= (mode == 1 ? 4 : 3); ++nf) {
                        if (nsub == 2 && n > 6) continue;
                        if (mode == 1 && nf == 4 && n > 6) continue;
                        CompiledDag D;
                        std::string e = compile_dag(n, nf, nsub, mode ? sig : nullptr, mode == 2, all != 0, 0, D);
                        if (!e.empty()) { printf("n=%d: %s\n", n, e.c_str()); return 1; }
                        total += D.n_states;
                        if (all && n >= 3) {                   // partial readout sets
                            CompiledDag P;
                            e = compile_dag(n, nf, nsub, mode ? sig : nullptr, mode == 2, true, (1u << 2) | (1u << n), P);
                            if (!e.empty()) { printf("orders n=%d: %s\n", n, e.c_str()); return 1; }
                            total += P.n_states;
                        }
                    }
    printf("ok, %llu states compiled\n", total);
    return 0;
}
