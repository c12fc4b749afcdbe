"""Seeded mixed-camera batches for the ragged tests (inputs only; none of the
method's arithmetic). A batch is built from dl0gen's camera models: each block
is one event of one telescope, blocks are laid out one after the other in a
flat uint16 buffer with optional junk gaps."""
from __future__ import annotations

import numpy as np

import dl0gen


class Batch:
    def __init__(self):
        self.tel_n_pixels, self.tel_n_samples, self.tel_W, self.tel_calib_offset = [], [], [], []
        self.blk_tel, self.blk_wf_offset, self.blk_out_offset = [], [], []
        self.pedestal = np.zeros(0, np.int32)
        self.gain = np.zeros(0, np.float32)
        self.wf = np.zeros(0, np.uint16)
        self.n_out = 0

    def tables(self):
        return (self.tel_n_pixels, self.tel_n_samples, self.tel_W, self.tel_calib_offset,
                self.blk_tel, self.blk_wf_offset, self.blk_out_offset)


def make_batch(tels, n_events, seed=0, gap=0, trigger=0.6, align=1, shuffle_out=False):
    """tels: list of (config name, number of telescopes of that camera) or of
    explicit (P, S, W) tuples. Every event triggers each telescope with
    probability ``trigger`` (at least one). ``gap`` junk samples may be inserted
    before a block (random 0..gap); ``align`` rounds block starts up to a
    multiple of that many samples."""
    rng = np.random.default_rng(seed)
    b = Batch()
    cams = []
    peds, gains = [], []
    cal = 0
    for spec, count in tels:
        for j in range(count):
            if isinstance(spec, str):
                c = dl0gen.CONFIGS[spec]
                P, S, W = c.n_pixels, c.n_samples, c.W
                ped, gain = dl0gen.calib(c)
                ped = (ped + rng.integers(-5, 6, P)).astype(np.int32)   # per-telescope calibration
                gain = (gain * np.float32(1.0 + 0.01 * j)).astype(np.float32)
            else:
                P, S, W = spec
                c = None
                ped = rng.integers(0, 600, P).astype(np.int32)
                gain = rng.uniform(0.9, 1.1, P).astype(np.float32)
            b.tel_n_pixels.append(P); b.tel_n_samples.append(S); b.tel_W.append(W)
            b.tel_calib_offset.append(cal)
            cal += P
            peds.append(ped); gains.append(gain)
            cams.append((c, P, S))
    b.pedestal = np.concatenate(peds)
    b.gain = np.concatenate(gains)
    chunks, pos, out = [], 0, 0
    for e in range(n_events):
        trig = [k for k in range(len(cams)) if rng.random() < trigger]
        if not trig:
            trig = [int(rng.integers(0, len(cams)))]
        for k in trig:
            c, P, S = cams[k]
            g = int(rng.integers(0, gap + 1)) if gap else 0
            start = pos + g
            start += -start % align
            if start > pos:
                chunks.append(rng.integers(0, 65536, start - pos).astype(np.uint16))
            if c is not None:
                blk = dl0gen.events_cpu(c, int(rng.integers(0, c.n_events)), 1)[0]
                # undo the shared calibration shift so the block sits on its own telescope's pedestal
                d = b.pedestal[b.tel_calib_offset[k]:b.tel_calib_offset[k] + P] - dl0gen.calib(c)[0]
                blk = np.clip(blk.astype(np.int64) + d[:, None], 0, 4095).astype(np.uint16)
            else:
                blk = rng.integers(0, 65536, (P, S)).astype(np.uint16)
            chunks.append(blk.ravel())
            b.blk_tel.append(k); b.blk_wf_offset.append(start); b.blk_out_offset.append(out)
            pos = start + P * S
            out += P
    b.wf = np.concatenate(chunks) if chunks else np.zeros(0, np.uint16)
    b.n_out = out
    if shuffle_out:                                  # same outputs, scattered block order
        sizes = [b.tel_n_pixels[k] for k in b.blk_tel]
        order = rng.permutation(len(sizes))
        offs, o = [0] * len(sizes), 0
        for i in order:
            offs[i] = o
            o += sizes[i]
        b.blk_out_offset = offs
    return b
