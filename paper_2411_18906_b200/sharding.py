"""Multi-GPU sharding of the hot path: chains (MC) and batch items (recount) are
independent, so they are split across ranks with NO data-path collective.  Results do not depend on the split because
the RNG is keyed by the GLOBAL chain id (hea_mc_run's chain0 argument)."""


def weak_chain_range(rank, chains_per_rank):
    """Weak scaling (bench.py): every rank runs `chains_per_rank` chains; returns (chain0, count)."""
    return rank * chains_per_rank, chains_per_rank


def strong_chain_range(rank, world, n_chains):
    """Strong scaling: n_chains global chains split as evenly as possible; returns (chain0, count)."""
    base, extra = divmod(n_chains, world)
    count = base + (1 if rank < extra else 0)
    chain0 = rank * base + min(rank, extra)
    return chain0, count
