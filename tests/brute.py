"""Pure-Python brute force (nested lists, element loops, no NumPy indexing) that pins the NumPy oracle.

Written independently from oracle/kv_migration.py, straight from the statement of the problem
(PAPER.md:134, :142, :237): a pool is pool[l][kv][b][e]; a stage copies, for every listed pair and
every layer and K|V, every element of the source block into the destination block.
"""


def pool_from_numpy(a):
    return [[[[int(a[l, kv, b, e]) for e in range(a.shape[3])] for b in range(a.shape[2])]
             for kv in range(2)] for l in range(a.shape[0])]


def copy_pool(p):
    return [[[list(blk) for blk in kvp] for kvp in lay] for lay in p]


def migrate_stage(src, src_ids, dst, dst_ids):
    assert len(src_ids) == len(dst_ids)
    n_layers = len(src)
    n_elems = len(src[0][0][0])
    for i in range(len(src_ids)):
        sb = int(src_ids[i])
        db = int(dst_ids[i])
        for l in range(n_layers):
            for kv in range(2):
                for e in range(n_elems):
                    dst[l][kv][db][e] = src[l][kv][sb][e]


def pack(src, src_ids):
    n_layers = len(src)
    n_elems = len(src[0][0][0])
    flat = []
    for i in range(len(src_ids)):
        for l in range(n_layers):
            for kv in range(2):
                for e in range(n_elems):
                    flat.append(src[l][kv][int(src_ids[i])][e])
    return flat


def unpack(flat, dst, dst_ids):
    n_layers = len(dst)
    n_elems = len(dst[0][0][0])
    p = 0
    for i in range(len(dst_ids)):
        for l in range(n_layers):
            for kv in range(2):
                for e in range(n_elems):
                    dst[l][kv][int(dst_ids[i])][e] = flat[p]
                    p += 1


def append_token(pool, table, t, block_size, token_elems, vals_of):
    b = int(table[t // block_size])
    s = t % block_size
    for l in range(len(pool)):
        for kv in range(2):
            v = vals_of(t, l, kv)
            for j in range(token_elems):
                pool[l][kv][b][s * token_elems + j] = int(v[j])


def attention(k_rows, v_rows, q, scale):
    """Textbook softmax attention for one head in Python floats. k_rows, v_rows: lists of lists."""
    import math
    s = [sum(qi * ki for qi, ki in zip(q, k)) * scale for k in k_rows]
    m = max(s)
    w = [math.exp(x - m) for x in s]
    z = sum(w)
    d = len(v_rows[0])
    return [sum(w[t] * v_rows[t][j] for t in range(len(w))) / z for j in range(d)]
