/*
 * hhrr_oracle_q19.c -- the fp64 CPU oracle on the paper's own velocity set, D3Q19 (Fig. 2 :107;
 * Table 1 :385-391 quotes its 152 / 204 B per cell on it).  TEST INFRASTRUCTURE ONLY, like hhrr_oracle.c, which
 * this translation unit instantiates with 19 directions: the 19 directions of D3Q27 with |c|^2 <= 2, weights
 * 1/3, 1/18, 1/36, and the third-order Hermite basis of the paper's ref. [43] (reading R23).
 * Built into its own library (libhhrr_oracle_q19.so); shares nothing with the CUDA path.
 */
#define OHRR_Q 19
#include "hhrr_oracle.c"
