// tu_elem_f64.cu -- instantiates the ELEMENTWISE kernels with one cosmology per redshift (cosmo_kernels.cuh: k_elem, k_elem_redo) for double.
#include "cosmo_kernels.cuh"

namespace cb {

template <bool kG>
static void elem_dispatch_f64(const ElemArgs& a, cudaStream_t st) {
    using T = double;
    const bool kT = a.which & (W_TL | W_AGE), kA = a.which & W_DABS;
    const dim3 grid((unsigned)cdiv64(a.N, CB_ELEM_BLOCK)), redo(148 * CB_REDO_GRID);      // second pass: persistent over a list whose length only the device knows
    if (kG) cudaMemsetAsync(a.redo_count, 0, sizeof(unsigned), st);
    const bool age = (a.which & W_AGE) != 0;
    if (kT && kA && age) { k_elem<T, true, true, kG, true><<<grid, CB_ELEM_BLOCK, 0, st>>>(a); if (kG) k_elem_redo<T, true, true, true><<<redo, ELEM_THREADS, 0, st>>>(a); }
    else if (kT && age) { k_elem<T, true, false, kG, true><<<grid, CB_ELEM_BLOCK, 0, st>>>(a); if (kG) k_elem_redo<T, true, false, true><<<redo, ELEM_THREADS, 0, st>>>(a); }
    else if (kT && kA) { k_elem<T, true, true, kG, false><<<grid, CB_ELEM_BLOCK, 0, st>>>(a); if (kG) k_elem_redo<T, true, true, true><<<redo, ELEM_THREADS, 0, st>>>(a); }
    else if (kT) { k_elem<T, true, false, kG, false><<<grid, CB_ELEM_BLOCK, 0, st>>>(a); if (kG) k_elem_redo<T, true, false, true><<<redo, ELEM_THREADS, 0, st>>>(a); }
    else if (kA) { k_elem<T, false, true, kG, false><<<grid, CB_ELEM_BLOCK, 0, st>>>(a); if (kG) k_elem_redo<T, false, true, true><<<redo, ELEM_THREADS, 0, st>>>(a); }
    else { k_elem<T, false, false, kG, false><<<grid, CB_ELEM_BLOCK, 0, st>>>(a); if (kG) k_elem_redo<T, false, false, true><<<redo, ELEM_THREADS, 0, st>>>(a); }
}

void launch_elem_f64(bool with_grad, const ElemArgs& a, cudaStream_t st) {
    if (with_grad) elem_dispatch_f64<true>(a, st);
    else elem_dispatch_f64<false>(a, st);
}

}  // namespace cb
