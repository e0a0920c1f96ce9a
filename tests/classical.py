"""Classical event-by-event coalescence (App. G.3) with an ordinary PRNG.

Independent pin for the oracle's coalescence semantics: same model, entirely different
mechanism (global state, explicit collision check, numpy Generator). Tiny inputs only. The global clock is
not simulated because species identities do not depend on it when the turnover rate is uniform (L2261-2263).
With non-uniform turnover the next lineage is picked proportionally to its cell's rate (rejection sampling,
L639)."""
import numpy as np


def simulate_classical(rng, start_locs, nu_of, disperse, rate_of=None):
    """start_locs: list of distinct hashable locations. nu_of(loc) -> speciation prob.
    disperse(rng, loc) -> parent location. Returns species label per lineage (arbitrary ints)."""
    n = len(start_locs)
    loc = list(start_locs)
    active = list(range(n))
    occupant = {l: i for i, l in enumerate(loc)}        # location -> active lineage
    parent = list(range(n))                             # union-find style pointer to the lineage merged into
    species = [-1] * n
    next_species = 0
    rmax = max(rate_of(l) for l in loc) if rate_of else 1.0
    while active:
        a = int(rng.integers(len(active)))
        i = active[a]
        if rate_of is not None:
            # rates change as lineages move: use a global bound supplied by the caller through rate_of.max
            if rng.random() * rate_of.max >= rate_of(loc[i]):
                continue
        if rng.random() < nu_of(loc[i]):
            species[i] = next_species; next_species += 1
            del occupant[loc[i]]
            active[a] = active[-1]; active.pop()
            continue
        new = disperse(rng, loc[i])
        if new == loc[i]:
            continue                                    # jumped onto itself: nothing changes
        del occupant[loc[i]]
        if new in occupant:                             # coalescence with the lineage living there (L2269-2274)
            parent[i] = occupant[new]
            active[a] = active[-1]; active.pop()
        else:
            loc[i] = new; occupant[new] = i
    out = []
    for i in range(n):
        r = i
        while species[r] < 0:
            r = parent[r]
        out.append(species[r])
    return out


def sad_of(labels):
    """species-abundance distribution: counts of species having abundance a (index a)."""
    _, counts = np.unique(labels, return_counts=True)
    return np.bincount(counts)


def simulate_classical_timed(rng, start_locs, nu, disperse_at, rate=1.0):
    """The same coalescence with the global clock simulated (uniform turnover `rate`): the n active lineages have events at total rate
    n * rate, so the time to the next event is Exp(n * rate). disperse_at(rng, loc, t) -> parent location
    for an event at time t (generations before the present): the landscape may depend on time (temporally varying habitat, L1498)."""
    n = len(start_locs)
    loc = list(start_locs)
    active = list(range(n))
    occupant = {l: i for i, l in enumerate(loc)}
    parent = list(range(n))
    species = [-1] * n
    next_species = 0
    t = 0.0
    while active:
        t += rng.exponential(1.0 / (rate * len(active)))
        a = int(rng.integers(len(active)))
        i = active[a]
        if rng.random() < nu:
            species[i] = next_species; next_species += 1
            del occupant[loc[i]]
            active[a] = active[-1]; active.pop()
            continue
        new = disperse_at(rng, loc[i], t)
        if new == loc[i]:
            continue
        del occupant[loc[i]]
        if new in occupant:
            parent[i] = occupant[new]
            active[a] = active[-1]; active.pop()
        else:
            loc[i] = new; occupant[new] = i
    out = []
    for i in range(n):
        r = i
        while species[r] < 0:
            r = parent[r]
        out.append(species[r])
    return out
