// k_packed_s2.cu -- streaming half-sweep kernel (packed layout), stream definition 2; see k_packed.inl
#define POTTS_ST 2
#include "k_packed.inl"
