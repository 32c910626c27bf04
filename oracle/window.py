"""The position-free window store as a deque (test infrastructure; see oracle/__init__.py).

"Making a chunk position-free changes the structure available: the same store can act as
a deque, evicting and admitting at either end of the window in O(1)".  "As the
oldest frame leaves, survivors re-rotate by the slide offset (free) and a later recall
rehydrates the dropped frame from the canonical store with a patch".

The paper fixes no page-allocation policy; the one below is reading R-13 of DESIGN.md and is
what makes block tables comparable bit-for-bit:

  * one global LIFO free list, initialised so that the first pops return pages 0, 1, 2, ...
  * admit pops n_tokens/P pages, in logical (token) order
  * evict pushes the chunk's pages back in REVERSE logical order (so an immediate re-admit
    of an equally long chunk gets the same pages in the same order)
  * logical token order of a request = deque order of its chunks
  * the first `n_pinned` chunks of a request (a text prefix, BASELINE.json config 4) are exempt
    from FRONT operations: FRONT means "just behind the pinned chunks"
  * position of chunk i = window_base + (tokens of chunks before it)
  * `phase` of a chunk = the RoPE position its keys currently sit at in the pool.
    materialize=1: every chunk whose position moved is re-rotated in place now
    (delta = position - phase, then phase = position).  materialize=0: nothing is touched;
    chunk_offset = position - phase is left for the decode kernel to apply on read.

This is the deliberately naive model: a Python list per request, positions recomputed from
scratch after every operation.
"""
FRONT, BACK = 0, 1


class Chunk:
    def __init__(self, handle, n_tokens, pages, phase):
        self.handle, self.n_tokens, self.pages, self.phase = handle, n_tokens, list(pages), phase


class WindowStore:
    def __init__(self, num_pages, page_size):
        self.P = page_size
        self.free = list(range(num_pages - 1, -1, -1))     # pop() -> 0, 1, 2, ...
        self.req = {}                                      # req -> dict(base, pinned, chunks)
        self.next_handle = 0

    # -- request lifetime ------------------------------------------------------------------
    def open(self, req, window_base=0):
        if req in self.req:
            raise RuntimeError("request already open")
        self.req[req] = {"base": int(window_base), "pinned": 0, "chunks": []}

    def pin(self, req, n_front_chunks):
        r = self.req[req]
        if not 0 <= n_front_chunks <= len(r["chunks"]):
            raise ValueError("cannot pin more chunks than the window holds")
        r["pinned"] = n_front_chunks

    def close(self, req):
        for c in reversed(self.req[req]["chunks"]):
            self.free.extend(reversed(c.pages))
        del self.req[req]

    # -- positions --------------------------------------------------------------------------
    def positions(self, req):
        r, pos, out = self.req[req], self.req[req]["base"], []
        for c in r["chunks"]:
            out.append(pos)
            pos += c.n_tokens
        return out

    def _settle(self, req, materialize):
        """After an op: list (handle, delta) of chunks to rotate in place now."""
        work = []
        if materialize:
            for c, pos in zip(self.req[req]["chunks"], self.positions(req)):
                if pos != c.phase:
                    work.append((c.handle, pos - c.phase))
                    c.phase = pos
        return work

    # -- the two deque operations -------------------------------------------------------------
    def admit(self, req, end, n_tokens, materialize=1):
        """Returns (handle, pages, p_target, rotations).  The admitted chunk itself is always
        materialised (relocate+patch to p_target, Eq. 1); `rotations` are the survivors."""
        r = self.req[req]
        if n_tokens <= 0 or n_tokens % self.P:
            raise ValueError("chunk length must be a positive multiple of the page size")
        need = n_tokens // self.P
        if need > len(self.free):
            raise MemoryError("no pages")
        pages = [self.free.pop() for _ in range(need)]
        c = Chunk(self.next_handle, n_tokens, pages, None)
        self.next_handle += 1
        idx = r["pinned"] if end == FRONT else len(r["chunks"])
        r["chunks"].insert(idx, c)
        c.phase = self.positions(req)[idx]
        return c.handle, pages, c.phase, self._settle(req, materialize)

    def evict(self, req, end, materialize=1):
        """Returns (handle, pages, rotations)."""
        r = self.req[req]
        if len(r["chunks"]) <= r["pinned"]:
            raise IndexError("window empty")
        idx = r["pinned"] if end == FRONT else len(r["chunks"]) - 1
        c = r["chunks"].pop(idx)
        self.free.extend(reversed(c.pages))
        return c.handle, c.pages, self._settle(req, materialize)

    # -- the linear view everything is compared through -----------------------------------------
    def export(self, req):
        r = self.req[req]
        bt, starts, offsets, handles = [], [0], [], []
        for c, pos in zip(r["chunks"], self.positions(req)):
            bt.extend(c.pages)
            starts.append(starts[-1] + c.n_tokens)
            offsets.append(pos - c.phase)
            handles.append(c.handle)
        slot = [bt[g // self.P] * self.P + g % self.P for g in range(starts[-1])]
        return {"block_table": bt, "slot_mapping": slot, "chunk_starts": starts,
                "chunk_offsets": offsets, "handles": handles, "positions": self.positions(req)}
