// Host harness of tests/test_symv_layout_host.py: csrc/symv_layout.h compiled with g++ (the CUDA qualifiers defined
// away), so that the layout of the reciprocity bank can be checked without a GPU.
#define __host__
#define __device__
#include "../paper_1910_07054_b200/csrc/symv_layout.h"

extern "C" {

// geometry of nz layers: out = {W, LW, EPW, nfull, half, NC, SPE, pairs per entry}
void hfft_test_symv_geom(int nz, long long* out) {
    const hfft::SymvGeom g = hfft::symv_geom(nz);
    out[0] = g.W; out[1] = g.LW; out[2] = g.EPW; out[3] = g.nfull; out[4] = g.half; out[5] = g.NC; out[6] = g.SPE;
    out[7] = hfft::symv_pairs_per_entry(g);
}

// position of the ordered pair (i, j): out = {couple, h, strip, transposed, float offset of component c for entry ent}
void hfft_test_symv_pos(int nz, int i, int j, int ent, int c, long long* out) {
    const hfft::SymvGeom g = hfft::symv_geom(nz);
    const hfft::SymvPos p = hfft::symv_pos(g, i, j);
    out[0] = p.couple; out[1] = p.h; out[2] = p.strip; out[3] = p.transposed;
    out[4] = hfft::symv_float_offset(g, p, ent, c);
}

}  // extern "C"
