// Test helper (CPU): prints the CUDA library's host-side tables (csrc/tables.hpp) so that
// tests/test_library_tables.py can pin them without a GPU.  Not part of the product.
#include <cstdio>
#include "../../paper_1907_08316_b200/csrc/tables.hpp"
int main() {
    for (int o = 1; o <= sldg::kMaxOrder; ++o) {
        double xi[8], w[8];
        sldg::gauss_legendre_01(o, xi, w);
        printf("GL %d", o);
        for (int j = 0; j < o; ++j) printf(" %.17g %.17g", xi[j], w[j]);
        printf("\n");
        std::vector<double> c = sldg::ab_polynomial_coefficients(o);
        printf("AB %d", o);
        for (double v : c) printf(" %.17g", v);
        printf("\n");
    }
    return 0;
}
