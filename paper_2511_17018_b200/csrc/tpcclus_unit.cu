// tpcclus_unit.cu -- one compilation unit of the device code (PAPER.md 64, section 3: one source file
// per kernel, compiled straight to a GPU binary, loaded with cuModuleLoad).  The build compiles this
// file once per unit with -DTPC_UNITS=<TPC_U_* bit> -cubin; the binaries are embedded in
// libtpcclus.so and loaded per handle (tpcclus.cu: load_unit).  Each unit gets the register
// allocation ptxas finds best for its kernels and its own __constant__ parameter block.
#ifndef TPC_UNITS
#error "compile with -DTPC_UNITS=<unit bit>"
#endif
#include "tpcclus_kernels.cuh"
