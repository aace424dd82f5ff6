// k_packed_s1.cu -- streaming half-sweep kernel (packed layout), stream definition 1; see k_packed.inl
#define POTTS_ST 1
#include "k_packed.inl"
