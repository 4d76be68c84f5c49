// art_decode_pc_kernel<G = 1, MODE, MT>: instantiations and launcher (see art_launch.h)
#define ART_PC_G 1
#include "art_pc_inst.inc"
