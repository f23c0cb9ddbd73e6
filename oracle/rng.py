"""Position-addressed uniforms for the oracle (TEST INFRASTRUCTURE).

The paper's draws come from "the per-request random number generator when available and
otherwise PyTorch's global generator" (§B.1.2) - not a reproducible
specification. BASELINE.json's north_star fixes "Gumbel-max on seeded uniforms supplied as
inputs". Reading R3: uniforms are *addressed by position*:
    u_sample[b, t, v]  -- step t = 1.. of sequence b, vocabulary id v
    u_switch[b, t]     -- t = 0 is the a_1 draw (Alg. 1 line 6, L346), t >= 1 the redraw after y_t
either given as explicit arrays or produced by the counter-based generator below, which the
CUDA side re-implements independently (no shared code):

    Philox-4x32-10 (Salmon et al., SC'11), key = (seed & 0xffffffff, seed >> 32),
    counter = (v >> 2, t, b, stream), stream 0 = sample, 1 = switch; output word v & 3.
    u = min((float32(r) + 0.5f) * 2^-32, 1 - 2^-24)  with IEEE round-to-nearest float32 ops.

u is never 0 and never 1, so `u < p` is never true at p = 0 and always true at p = 1.
The Gumbel variate is g = -ln(-log1p(-u)) (E = -log1p(-u) is a unit exponential; this
orientation keeps full relative resolution for the small-E winners among ~150k ids).
"""
import numpy as np

_M0 = np.uint64(0xD2511F53)
_M1 = np.uint64(0xCD9E8D57)
_W0 = np.uint32(0x9E3779B9)
_W1 = np.uint32(0xBB67AE85)
_MASK32 = np.uint64(0xFFFFFFFF)

STREAM_SAMPLE = 0
STREAM_SWITCH = 1


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox-4x32 with 10 rounds. Inputs broadcastable uint32 arrays; returns 4 uint32 arrays.

    Round (Salmon et al. 2011, Fig. 3 / Random123 philox.h): (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2,
    c <- (hi1 ^ c1 ^ k0, lo1, hi0 ^ c3 ^ k1, lo0); key bumped by the Weyl constants between rounds.
    """
    c0, c1, c2, c3, k0, k1 = np.broadcast_arrays(*[np.asarray(a, dtype=np.uint32) for a in (c0, c1, c2, c3, k0, k1)])
    c0 = c0.copy(); c1 = c1.copy(); c2 = c2.copy(); c3 = c3.copy(); k0 = k0.copy(); k1 = k1.copy()
    with np.errstate(over="ignore"):
        for r in range(10):
            p0 = _M0 * c0.astype(np.uint64)
            p1 = _M1 * c2.astype(np.uint64)
            hi0 = (p0 >> np.uint64(32)).astype(np.uint32)
            lo0 = (p0 & _MASK32).astype(np.uint32)
            hi1 = (p1 >> np.uint64(32)).astype(np.uint32)
            lo1 = (p1 & _MASK32).astype(np.uint32)
            n0 = hi1 ^ c1 ^ k0
            n1 = lo1
            n2 = hi0 ^ c3 ^ k1
            n3 = lo0
            c0, c1, c2, c3 = n0, n1, n2, n3
            if r < 9:
                k0 = (k0 + _W0).astype(np.uint32)
                k1 = (k1 + _W1).astype(np.uint32)
    return c0, c1, c2, c3


def uniform_from_bits(r):
    """uint32 -> float32 in (0, 1): min((float32(r) + 0.5f) * 2^-32, 1 - 2^-24), each op rounded to float32."""
    r = np.asarray(r, dtype=np.uint32)
    f = r.astype(np.float32)                       # round-to-nearest-even conversion
    f = (f + np.float32(0.5)).astype(np.float32)
    f = (f * np.float32(2.0 ** -32)).astype(np.float32)
    return np.minimum(f, np.float32(1.0 - 2.0 ** -24)).astype(np.float32)


def _key(seed):
    seed = int(seed) & 0xFFFFFFFFFFFFFFFF
    return np.uint32(seed & 0xFFFFFFFF), np.uint32(seed >> 32)


def uniforms_sample(seed, b, t, vocab):
    """u_sample[b, t, 0:vocab] as float32 (stream 0)."""
    k0, k1 = _key(seed)
    nblk = (vocab + 3) // 4
    blk = np.arange(nblk, dtype=np.uint32)
    w = philox4x32_10(blk, np.uint32(t), np.uint32(b), np.uint32(STREAM_SAMPLE), k0, k1)
    bits = np.stack(w, axis=1).reshape(-1)[:vocab]
    return uniform_from_bits(bits)


def uniforms_switch(seed, b, t):
    """u_switch[b, t] as float32 (stream 1, block 0, word 0)."""
    k0, k1 = _key(seed)
    w = philox4x32_10(np.uint32(0), np.uint32(t), np.uint32(b), np.uint32(STREAM_SWITCH), k0, k1)
    return np.float32(uniform_from_bits(w[0]))


def gumbel_from_uniform(u):
    """g = -ln(E), E = -log1p(-u): standard Gumbel variate from a uniform in (0,1). float64 math
    on the exact float32 value of u (BASELINE.json north_star (g): Gumbel-max on supplied uniforms)."""
    u = np.asarray(u, dtype=np.float64)
    return -np.log(-np.log1p(-u))
