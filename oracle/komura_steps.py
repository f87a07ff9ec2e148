"""The paper's four steps, written out step by step on an NN list.  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Pure Python, for small cases only.  Follows PAPER.md section 3 (lines 111-149) in the paper's order and notation:

  (i)   initialization  -- residual list = neighbours numbered lower than the site; label[i] = the lowest of them
                           (removed from the list), else i                       (Fig. 2 at :63-77)
  (ii)  analysis        -- label[i] <- label[label[i]] until unchanged            (Fig. 3 left at :79-93)
  (iii) label reduction -- every site runs Algorithm 1 over its residual list
  (iv)  analysis        -- again                                                  (Fig. 4 at :95-109)

Algorithm 1's last lines are flattened in the source text.  Reading R3 of DESIGN.md is used:

    label_3 <- atomicMin(&label[label_1], label_2)
    if   label_3 == label_2: flag <- true
    elif label_3 >  label_2: label_1 <- label_3
    else (label_3 < label_2): label_1 <- label_2; label_2 <- label_3

`reduction_threads` expresses step (iii) as one generator per site that yields before every access to `label`, so
a test can interleave the "threads" arbitrarily (the GPU runs them concurrently; the final labels must not depend
on the schedule).  `alt_reading=True` switches to the rejected reading of the garbled lines (the trailing
`label_2 <- label_3` taken as unconditional), which tests show to be wrong.
"""
import random


def initialization(nn_list):
    """Step (i).  nn_list[i] = iterable of i's neighbours.  Returns (label, residual)."""
    n = len(nn_list)
    label = list(range(n))
    residual = []
    for i in range(n):
        lower = sorted(j for j in nn_list[i] if j < i)
        if lower:
            label[i] = lower[0]
            lower = lower[1:]
        residual.append(lower)
    return label, residual


def analysis(label):
    """Steps (ii)/(iv): every site follows label[label[...]] until it stops changing (reading R2: per-site chase)."""
    n = len(label)
    out = list(label)
    for i in range(n):
        l = label[i]
        while l != label[l]:
            l = label[l]
        out[i] = l
    return out


def _algorithm1(label, i, j, alt_reading=False):
    """Algorithm 1 for the pair (site i, residual entry j) as a generator: yields before each access to label[]."""
    yield
    label_1 = label[i]
    while True:
        yield
        nxt = label[label_1]
        if label_1 == nxt:
            break
        label_1 = nxt
    yield
    label_2 = label[j]
    while True:
        yield
        nxt = label[label_2]
        if label_2 == nxt:
            break
        label_2 = nxt
    flag = True
    if label_1 != label_2:
        flag = False
    if label_1 < label_2:
        label_1, label_2 = label_2, label_1
    while not flag:
        yield
        label_3 = label[label_1]                      # atomicMin(&label[label_1], label_2): returns the old value
        if label_2 < label_3:
            label[label_1] = label_2
        if label_3 == label_2:
            flag = True
        elif label_3 > label_2:
            label_1 = label_3
        else:
            label_1 = label_2
            if not alt_reading:
                label_2 = label_3
        if alt_reading:
            label_2 = label_3                         # rejected reading: trailing statement taken as unconditional


def _site_thread(label, i, residual_i, alt_reading):
    for j in residual_i:
        yield from _algorithm1(label, i, j, alt_reading)


def label_reduction(label, residual, schedule_seed=None, alt_reading=False, max_steps=10_000_000):
    """Step (iii), in place.  schedule_seed=None: sites in ascending order, one after the other;
    otherwise the site "threads" are interleaved at memory-access granularity by a seeded scheduler."""
    n = len(label)
    threads = [_site_thread(label, i, residual[i], alt_reading) for i in range(n) if residual[i]]
    if schedule_seed is None:
        for t in threads:
            for _ in t:
                pass
        return label
    rng = random.Random(schedule_seed)
    steps = 0
    while threads:
        k = rng.randrange(len(threads))
        try:
            next(threads[k])
        except StopIteration:
            threads[k] = threads[-1]
            threads.pop()
        steps += 1
        if steps > max_steps:
            raise RuntimeError("label reduction did not terminate")
    return label


def four_steps(nn_list, schedule_seed=None, alt_reading=False):
    """All four steps; returns the states after (i), (ii), (iii), (iv)."""
    label, residual = initialization(nn_list)
    after_i = list(label)
    after_ii = analysis(label)
    label = list(after_ii)
    label_reduction(label, residual, schedule_seed, alt_reading)
    after_iii = list(label)
    after_iv = analysis(label)
    return after_i, after_ii, after_iii, after_iv


def nn_list_from_bonds(n_sites, bonds):
    """NN list of an undirected bond list; self-loops dropped, duplicates kept once."""
    nn = [set() for _ in range(n_sites)]
    for u, v in bonds:
        if u != v:
            nn[u].add(v)
            nn[v].add(u)
    return [sorted(s) for s in nn]
