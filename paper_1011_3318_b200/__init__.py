"""wcras: RAS-preconditioned mixed-precision nested BiCGStab for the Wilson-clover Dirac equation on one
B200 (arXiv:1011.3318 hot path).  `binding` wraps the C ABI of libwcras.so (include/wcras.h); `inputs`
holds the seeded synthetic input generators (no method arithmetic); `build` compiles the library."""
