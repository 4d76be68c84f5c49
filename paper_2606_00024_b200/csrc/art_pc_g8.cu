// art_decode_pc_kernel<G = 8, MODE, MT>: instantiations and launcher (see art_launch.h)
#define ART_PC_G 8
#include "art_pc_inst.inc"
