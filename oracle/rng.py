"""Counter-based random draws for the SVI / HMC consumers, numpy restatement.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  The paper draws its random numbers inside TFP/JAX (PAPER.md L89-100:
"n_VI draws per step"; L340: TFP's HMC) and prints no generator; the task's rule is that either the draws are inputs
(gl_svi_step / gl_hmc_step take them) or both sides implement the same counter-based generator.  This is that generator
(reading S22):

  bits     Philox4x32-10 (Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3", SC'11): 10 rounds of
           (c0,c1,c2,c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0)), key bumped by the Weyl
           constants between rounds.
  key      (seed low word, seed high word)
  counter  (step low word, step high word, row index i, stream_id * 2^24 + block), block = j // 4 for element j of a row
  uniform  u = (word + 0.5) * 2^-32 in fp64: never 0 or 1
  normal   Box-Muller in fp64 on the word pairs (0,1) and (2,3) of one block: r = sqrt(-2 ln u_a), phi = 2 pi u_b,
           elements 4 block + (0,1,2,3) = (r cos phi, r sin phi) of pair (0,1), then of pair (2,3); rounded to fp32
  log u    ln of the uniform from word 0 of block 0, rounded to fp32
"""
import numpy as np

M0, M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
W0, W1 = 0x9E3779B9, 0xBB67AE85
MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(counter, key):
    """counter [..., 4], key [..., 2] (integers < 2^32) -> [..., 4] uint32 words."""
    c = [np.asarray(counter)[..., i].astype(np.uint64) for i in range(4)]
    k = [np.asarray(key)[..., i].astype(np.uint64) for i in range(2)]
    for r in range(10):
        if r > 0:
            k = [(k[0] + np.uint64(W0)) & MASK, (k[1] + np.uint64(W1)) & MASK]
        p0 = M0 * c[0]; p1 = M1 * c[2]                      # < 2^64: exact in uint64
        hi0, lo0 = p0 >> np.uint64(32), p0 & MASK
        hi1, lo1 = p1 >> np.uint64(32), p1 & MASK
        c = [hi1 ^ c[1] ^ k[0], lo1, hi0 ^ c[3] ^ k[1], lo0]
    return np.stack(c, axis=-1).astype(np.uint32)


def _words(seed, step, stream_id, n_rows, n_blocks):
    seed, step = int(seed), int(step)
    assert 0 <= stream_id < 256 and n_blocks <= 1 << 24
    i = np.arange(n_rows, dtype=np.uint64)[:, None]
    b = np.arange(n_blocks, dtype=np.uint64)[None, :]
    ctr = np.empty((n_rows, n_blocks, 4), dtype=np.uint64)
    ctr[..., 0] = step & 0xFFFFFFFF; ctr[..., 1] = (step >> 32) & 0xFFFFFFFF
    ctr[..., 2] = i; ctr[..., 3] = np.uint64(stream_id << 24) + b
    key = np.empty((n_rows, n_blocks, 2), dtype=np.uint64)
    key[..., 0] = seed & 0xFFFFFFFF; key[..., 1] = (seed >> 32) & 0xFFFFFFFF
    return philox4x32_10(ctr, key)


def uniform_of(words):
    return (words.astype(np.float64) + 0.5) * 2.0 ** -32


def draw_normal(seed, step, stream_id, n_rows, n_cols):
    """[n_rows][n_cols] fp32 standard normals."""
    nb = (n_cols + 3) // 4
    u = uniform_of(_words(seed, step, stream_id, n_rows, nb))          # [n, nb, 4]
    out = np.empty((n_rows, nb, 4))
    for a in (0, 2):
        r = np.sqrt(-2.0 * np.log(u[..., a])); phi = 2.0 * np.pi * u[..., a + 1]
        out[..., a] = r * np.cos(phi); out[..., a + 1] = r * np.sin(phi)
    return out.reshape(n_rows, nb * 4)[:, :n_cols].astype(np.float32)


def draw_log_uniform(seed, step, stream_id, n_rows):
    """[n_rows] fp32: ln u, u uniform on (0, 1)."""
    u = uniform_of(_words(seed, step, stream_id, n_rows, 1))[:, 0, 0]
    return np.log(u).astype(np.float32)
