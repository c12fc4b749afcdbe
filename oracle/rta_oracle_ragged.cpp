// oracle/rta_oracle_ragged.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain single-threaded CPU definition of extraction over a mixed-camera batch
// (SURVEY.md §8(f) NEXT-3). The paper's array has three telescope sizes
// (§1), operates in "multiple sub-array" configurations
// (§2.2) and its Central Event Builder merges the data of the
// telescopes triggered by the same event (§4.1); it gives no layout
// for such a merged event. The layout below is the builder's (DESIGN.md
// readings R28-R30):
//
//   telescope k (k = 0 .. n_tel-1) has a camera of tel_n_pixels[k] pixels read
//   out with tel_n_samples[k] samples per trace, is extracted with window
//   tel_W[k], and owns the calibration pedestal[tel_calib_offset[k] + p],
//   gain[tel_calib_offset[k] + p], p = 0 .. tel_n_pixels[k]-1.
//
//   block b (b = 0 .. n_blocks-1) is the readout of telescope blk_tel[b] for one
//   event: a dense uint16 [n_pixels][n_samples] array starting at sample index
//   blk_wf_offset[b] of the waveform buffer. Its results go to the flat output
//   index blk_out_offset[b] + p. Blocks may come in any order, with gaps between
//   them in either buffer.
//
// What is computed per trace is exactly the sliding-window definition of
// oracle/rta_oracle.cpp (BASELINE.json:north_star sentence 2), block by block,
// in block order; nothing is fused or reordered.
//
// Shares no code with paper_1307_6489_b200/csrc. Parity status: pinned
// (tests/test_oracle_ragged_pins.py): a hand-assembled mixed batch of hand-worked
// traces (tests/golden/ragged.json), an independent numpy restatement per block,
// closed forms per block, block-order and gap invariance, reduction of a uniform
// batch to the pinned uniform oracle.
#include <cstddef>
#include <cstdint>

extern "C" int rta_oracle_extract(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                                  int32_t n_samples, const int32_t* pedestal, const float* gain,
                                  int32_t W, int32_t* out_sum, int32_t* out_start,
                                  float* out_charge, float* out_time);

extern "C" {

// Returns 0 on success, 1 on a bad table (telescope index out of range, bad
// shape, negative offset).
int rta_oracle_extract_ragged(const uint16_t* wf, int32_t n_tel, const int32_t* tel_n_pixels,
                              const int32_t* tel_n_samples, const int32_t* tel_W,
                              const int64_t* tel_calib_offset, int64_t n_blocks,
                              const int32_t* blk_tel, const int64_t* blk_wf_offset,
                              const int64_t* blk_out_offset, const int32_t* pedestal,
                              const float* gain, int32_t* out_sum, int32_t* out_start,
                              float* out_charge, float* out_time) {
  if (n_tel < 0 || n_blocks < 0) return 1;
  for (int64_t b = 0; b < n_blocks; ++b) {
    const int32_t k = blk_tel[b];
    if (k < 0 || k >= n_tel) return 1;
    if (blk_wf_offset[b] < 0 || blk_out_offset[b] < 0 || tel_calib_offset[k] < 0) return 1;
  }
  for (int64_t b = 0; b < n_blocks; ++b) {
    const int32_t k = blk_tel[b];
    const int64_t o = blk_out_offset[b];
    const int64_t c = tel_calib_offset[k];
    // one block = one event of telescope k's camera
    const int rc = rta_oracle_extract(wf + blk_wf_offset[b], 1, tel_n_pixels[k], tel_n_samples[k],
                                      pedestal + c, gain + c, tel_W[k], out_sum + o,
                                      out_start + o, out_charge + o, out_time + o);
    if (rc != 0) return 1;
  }
  return 0;
}

}  // extern "C"
