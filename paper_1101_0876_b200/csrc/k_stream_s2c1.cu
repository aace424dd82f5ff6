// k_stream_s2c1.cu -- streaming half-sweep kernel (U8), stream definition 2, colour 1; see k_stream.inl
#define POTTS_ST 2
#define POTTS_COLOUR 1
#include "k_stream.inl"
