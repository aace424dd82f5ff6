// k_stream_s2c0.cu -- streaming half-sweep kernel (U8), stream definition 2, colour 0; see k_stream.inl
#define POTTS_ST 2
#define POTTS_COLOUR 0
#include "k_stream.inl"
