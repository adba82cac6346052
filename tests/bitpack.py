"""Test helper: (.., L, L) {0,1} arrays <-> the ABI's bit-packed (.., L, W) uint32 words
(include/tnmc.h: bit c%32 of word c/32 is 1 iff s(r,c) = +1).  Pure data movement."""
import numpy as np


def pack(cfg):
    cfg = np.asarray(cfg).astype(np.uint32)
    L = cfg.shape[-1]
    W = (L + 31) // 32
    pad = np.zeros(cfg.shape[:-1] + (W * 32,), dtype=np.uint32)
    pad[..., :L] = cfg
    pad = pad.reshape(cfg.shape[:-1] + (W, 32))
    return (pad << np.arange(32, dtype=np.uint32)).sum(axis=-1, dtype=np.uint64).astype(np.uint32)


def unpack(words, L):
    words = np.asarray(words).astype(np.uint32)
    bits = (words[..., :, None] >> np.arange(32, dtype=np.uint32)) & 1
    return bits.reshape(words.shape[:-1] + (-1,))[..., :L].astype(np.int8)
