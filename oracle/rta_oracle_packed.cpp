// oracle/rta_oracle_packed.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain single-threaded CPU definition of the packed-sample ingest
// (SURVEY.md §8(f) NEXT-2). The paper sends DL0 data as "a logical sequence of
// bits ... according with the definition of the satellite telemetry [12]"
// (§5) and says nothing else about the format; refs [11], [12]
// are not available. The format below is therefore the
// builder's (readings R25-R27), chosen for 12-bit digitisers
// (BASELINE.json:configs: "uint16 12-bit clamped [0,4095]"):
//
//   "P12": the dense sample stream wf[e][p][s] (sample fastest, no headers, no
//   per-trace or per-event padding), flat sample index n = (e*P + p)*S + s, is
//   stored 12 bits per sample, little-endian in bits: sample n occupies bits
//   [12 n, 12 n + 12) of the byte stream, bit b of the stream being bit (b % 8)
//   of byte (b / 8). Equivalently, for every pair a = sample 2k, b = sample 2k+1:
//       byte 3k   =  a        & 0xFF
//       byte 3k+1 = (a >> 8)  | ((b & 0xF) << 4)
//       byte 3k+2 =  b >> 4
//   The stream holds ceil(12 N / 8) bytes for N samples; when N is odd the high
//   nibble of the last byte is padding and is ignored.
//
// Decoding is exact (an encoding, not an approximation): the oracle follows
// the bit definition literally, one bit at a time. Extraction from a packed
// stream is "decode, then the sliding-window definition" (oracle/rta_oracle.cpp),
// nothing fused.
//
// Shares no code with paper_1307_6489_b200/csrc or with dl0gen's encoder.
// Parity status: pinned (tests/test_oracle_packed_pins.py): hand-worked byte
// fixtures (tests/golden/packed12.json), numpy unpackbits restatement, every
// 12-bit value at both nibble phases, closed-form byte patterns.
#include <cstddef>
#include <cstdint>
#include <vector>

extern "C" int rta_oracle_extract(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                                  int32_t n_samples, const int32_t* pedestal, const float* gain,
                                  int32_t W, int32_t* out_sum, int32_t* out_start,
                                  float* out_charge, float* out_time);

extern "C" {

// out[n] = sample n of the P12 stream, n = 0 .. n_total-1 (bit by bit).
int rta_oracle_unpack12(const uint8_t* packed, int64_t n_total, uint16_t* out) {
  if (n_total < 0) return 1;
  for (int64_t n = 0; n < n_total; ++n) {
    unsigned v = 0;
    for (int i = 0; i < 12; ++i) {
      const int64_t bit = 12 * n + i;
      const unsigned b = (packed[bit / 8] >> (bit % 8)) & 1u;
      v |= b << i;
    }
    out[n] = (uint16_t)v;
  }
  return 0;
}

// Sliding-window extraction (BASELINE.json:north_star sentence 2) of a P12 stream.
int rta_oracle_extract_packed12(const uint8_t* packed, int64_t n_events, int32_t n_pixels,
                                int32_t n_samples, const int32_t* pedestal, const float* gain,
                                int32_t W, int32_t* out_sum, int32_t* out_start,
                                float* out_charge, float* out_time) {
  if (n_events < 0 || n_pixels < 1 || n_samples < 1) return 1;
  const int64_t n_total = n_events * (int64_t)n_pixels * (int64_t)n_samples;
  std::vector<uint16_t> wf((size_t)n_total);
  if (rta_oracle_unpack12(packed, n_total, wf.data()) != 0) return 1;
  return rta_oracle_extract(wf.data(), n_events, n_pixels, n_samples, pedestal, gain, W, out_sum,
                            out_start, out_charge, out_time);
}

}  // extern "C"
