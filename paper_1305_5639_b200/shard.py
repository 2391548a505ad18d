"""Channel sharding of the X-engine across processes -- host logic only.

Eq. 2 is independent per frequency channel (the paper's own "orthogonal correlation triangles separating
frequency channels"), so rank r of `world` ranks can own a contiguous block of channels, run its own
corr_xengine on `in[:, c0:c1]` and write its own slab `out[c0:c1]`: no data-path collective, disjoint outputs.
BASELINE.json's north_star runs on ONE GPU, so `bench.py` uses this only under the optional `--shard channels`.
"""


def channel_range(n_chan, world, rank):
    """[c0, c1) of rank `rank`: contiguous blocks whose sizes differ by at most one, in rank order, covering [0, n_chan)."""
    if world < 1 or not 0 <= rank < world or n_chan < 0:
        raise ValueError("bad sharding arguments")
    base, extra = divmod(n_chan, world)
    c0 = rank * base + min(rank, extra)
    return c0, c0 + base + (1 if rank < extra else 0)
