// CPU TEST HARNESS (tests only): compiles the generated per-(event, helicity) device functions with g++
// so that the emitted diagram program and the helas.cuh routines can be checked against the oracle
// without a GPU.  Never linked into the product library.
#include "../paper_2510_05392_b200/csrc/generated/gg_ttx_jamps.cuh"
#include "../paper_2510_05392_b200/csrc/generated/gg_ttxg_jamps.cuh"
#include "../paper_2510_05392_b200/csrc/generated/gg_ttxgg_jamps.cuh"
#ifdef WITH_GGTTGGG
#include "../paper_2510_05392_b200/csrc/generated/gg_ttxggg_jamps.cuh"
#endif

template <typename T, typename F>
static void run(F f, int ncolor, const double* pe, int ihel, double mt, double wt, double* out)
{
    mg::cx<T>* j = new mg::cx<T>[ncolor];
    f(pe, ihel, T(mt), T(wt), j);
    for (int c = 0; c < ncolor; c++) { out[2 * c] = j[c].re; out[2 * c + 1] = j[c].im; }
    delete[] j;
}

extern "C" int host_jamps(int ngluon, int use_float, const double* pe, int ihel, double mt, double wt, double* out)
{
#define CASE(N, NS)                                                                                   \
    if (ngluon == N) {                                                                                \
        if (use_float) run<float>(mg::NS::jamps<float>, mg::NS::NCOLOR, pe, ihel, mt, wt, out);       \
        else run<double>(mg::NS::jamps<double>, mg::NS::NCOLOR, pe, ihel, mt, wt, out);               \
        return mg::NS::NCOLOR;                                                                        \
    }
    CASE(2, gg_ttx)
    CASE(3, gg_ttxg)
    CASE(4, gg_ttxgg)
#ifdef WITH_GGTTGGG
    CASE(5, gg_ttxggg)
#endif
    return -1;
}
