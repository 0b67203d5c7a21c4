"""TEST INFRASTRUCTURE -- oracle of the bounded entity cache.

PAPER.md L43: detected entities go through an "LRU cache to amortise repeated lookups across records"; L50 / L52: the
pseudonym of an entity is HMAC-SHA256(key, entity) and never changes.  The paper gives neither a capacity nor the
granularity of "recently used", so this build fixes reading D21:

  * recency is call-granular: a call to `pseudonymize` (one batch of spans) stamps every entity it looks up -- hit or new --
    with the call's sequence number 1, 2, 3, ...;
  * `evict(keep)` keeps the `keep` entries with the largest stamps; inside the cut-off stamp the lowest uids stay; survivors
    are renumbered 0..keep-1 in their old uid order and keep bytes, digest and stamp; hit / lookup counters are untouched;
  * inside one call spans are processed in order: the first occurrence of an unknown entity is a miss (hit = 0) and gets
    uid = number of entries before it, every later occurrence is a hit -- as in oracle/crypto.py.

Plain Python: a dict in insertion order plus `hmac` from the standard library as the HMAC step.  Pins:
tests/test_oracle_cache_lru.py (hand-worked trace; with one span per call and an eviction after every call the hit / miss
sequence is a textbook LRU, checked against collections.OrderedDict; pseudonyms do not depend on evictions).
"""
import hashlib
import hmac


class LruCache:
    def __init__(self, key):
        self.key = bytes(key)
        self.entries = {}            # entity bytes -> [uid, digest, stamp]; dict order = uid order
        self.epoch = 0
        self.n_lookups = 0
        self.n_hits = 0

    def pseudonymize(self, spans):
        """spans: list of bytes.  Returns (hit flags, uids, digests) per span."""
        self.epoch += 1
        hit, uid, dig = [], [], []
        for e in spans:
            e = bytes(e)
            ent = self.entries.get(e)
            if ent is None:
                ent = [len(self.entries), hmac.new(self.key, e, hashlib.sha256).digest(), self.epoch]
                self.entries[e] = ent
                hit.append(0)
            else:
                ent[2] = self.epoch
                hit.append(1)
            uid.append(ent[0])
            dig.append(ent[1])
        self.n_lookups += len(spans)
        self.n_hits += sum(hit)
        return hit, uid, dig

    def evict(self, keep):
        """Returns the number of entries dropped."""
        n = len(self.entries)
        if keep >= n:
            return 0
        order = sorted(self.entries.items(), key=lambda kv: (-kv[1][2], kv[1][0]))[:keep]     # newest stamps, then lowest uid
        order.sort(key=lambda kv: kv[1][0])                                                   # back to uid order
        self.entries = {}
        for new_uid, (e, ent) in enumerate(order):
            self.entries[e] = [new_uid, ent[1], ent[2]]
        return n - keep

    def export(self):
        """[(entity bytes, digest)] in uid order."""
        return [(e, ent[1]) for e, ent in self.entries.items()]
