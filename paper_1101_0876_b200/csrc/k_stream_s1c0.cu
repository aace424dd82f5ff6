// k_stream_s1c0.cu -- streaming half-sweep kernel (U8), stream definition 1, colour 0; see k_stream.inl
#define POTTS_ST 1
#define POTTS_COLOUR 0
#include "k_stream.inl"
