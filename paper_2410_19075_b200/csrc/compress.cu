// COMPRESS of Algorithm 2 on the host, on position sets instead of bit vectors:
//   V <- L_0;  for every row i:  d = XOR(ROL(L_i, i), V);  C_i <- index of d in the table D
// (ROL moves the bit at position j to (j - i) mod n, "addition of bits' positions modulo N",
// PAPER.md:173; XOR of two sorted position lists is their merge without the common elements).
// Done once per matrix, as in the paper; the table lookup FIND(D_j == d) is a hash of the
// positions followed by a full comparison, so the expected cost is O(nnz).
// Host code only (no kernel here); EXTRACT runs on the device inside the stage kernels
// (models.cuh: for_each_neighbor<NET_TOPO_COMPRESSED>).
#include <stdlib.h>

#include <algorithm>
#include <new>
#include <unordered_map>
#include <vector>

#include "oscnet_internal.cuh"

namespace {

struct Storage {
    std::vector<int32_t> v, dpos, c;
    std::vector<int64_t> dptr;
};
// standard-layout: a pointer to `pub` (what the caller holds) is a pointer to the Owned
struct Owned {
    net_compressed pub;
    Storage* st;
};

uint64_t hash_positions(const std::vector<int32_t>& d) {
    uint64_t hsh = 0xcbf29ce484222325ULL ^ (uint64_t)d.size();
    for (int32_t p : d) { hsh ^= (uint64_t)(uint32_t)p; hsh *= 0x100000001b3ULL; hsh ^= hsh >> 29; }
    return hsh;
}

}  // namespace

#pragma GCC visibility push(default)
extern "C" {

int32_t net_compress_csr(int64_t n, const int64_t* row_ptr, const int32_t* col_idx, net_compressed** out) {
    using oscnet::set_err;
    if (!out) return set_err(nullptr, NET_ERR_INVALID, "out is NULL");
    *out = nullptr;
    if (n < 1 || n > 2147483647LL || !row_ptr || (row_ptr[n] > 0 && !col_idx))
        return set_err(nullptr, NET_ERR_INVALID, "net_compress_csr: bad n or NULL arrays");
    Owned* owned = new (std::nothrow) Owned;
    Storage* o = new (std::nothrow) Storage;
    if (!owned || !o) { delete owned; delete o; return set_err(nullptr, NET_ERR_INVALID, "out of host memory"); }
    owned->st = o;
    auto drop = [&]() { delete o; delete owned; };
    try {
        std::vector<int32_t> shifted, d;
        auto rol = [&](int64_t i) {              // ROL(L_i, i) as a sorted position list
            shifted.clear();
            for (int64_t e = row_ptr[i]; e < row_ptr[i + 1]; ++e) {
                const int64_t j = col_idx[e];
                if (j < 0 || j >= n) return false;
                int64_t p = j - i;
                if (p < 0) p += n;
                shifted.push_back((int32_t)p);
            }
            std::sort(shifted.begin(), shifted.end());
            shifted.erase(std::unique(shifted.begin(), shifted.end()), shifted.end());
            return true;
        };
        if (row_ptr[0] != 0) { drop(); return set_err(nullptr, NET_ERR_TOPOLOGY, "net_compress_csr: row_ptr[0] != 0"); }
        if (!rol(0)) { drop(); return set_err(nullptr, NET_ERR_TOPOLOGY, "net_compress_csr: index outside [0, n)"); }
        o->v = shifted;                          // V <- L_0
        o->c.resize((size_t)n);
        o->dptr.push_back(0);
        std::unordered_multimap<uint64_t, int32_t> index;
        for (int64_t i = 0; i < n; ++i) {
            if (row_ptr[i + 1] < row_ptr[i]) { drop(); return set_err(nullptr, NET_ERR_TOPOLOGY, "net_compress_csr: row_ptr not monotone"); }
            if (!rol(i)) { drop(); return set_err(nullptr, NET_ERR_TOPOLOGY, "net_compress_csr: index outside [0, n)"); }
            d.clear();                           // d = XOR(ROL(L_i, i), V)
            std::set_symmetric_difference(shifted.begin(), shifted.end(), o->v.begin(), o->v.end(), std::back_inserter(d));
            const uint64_t key = hash_positions(d);
            int32_t found = -1;                  // FIND(D_j == d)
            auto range = index.equal_range(key);
            for (auto it = range.first; it != range.second && found < 0; ++it) {
                const int64_t b = o->dptr[it->second], e = o->dptr[it->second + 1];
                if (e - b == (int64_t)d.size() && std::equal(d.begin(), d.end(), o->dpos.begin() + b)) found = it->second;
            }
            if (found < 0) {                     // append to the table
                found = (int32_t)(o->dptr.size() - 1);
                o->dpos.insert(o->dpos.end(), d.begin(), d.end());
                o->dptr.push_back((int64_t)o->dpos.size());
                index.emplace(key, found);
            }
            o->c[(size_t)i] = found;
        }
    } catch (...) {
        drop();
        return set_err(nullptr, NET_ERR_INVALID, "net_compress_csr: out of host memory");
    }
    if (o->dpos.empty()) o->dpos.push_back(0);   // keep data() non-null
    net_compressed& pub = owned->pub;
    pub.v_len = (int64_t)o->v.size();
    if (o->v.empty()) o->v.push_back(0);         // keep data() non-null
    pub.n = n;
    pub.v_pos = o->v.data();
    pub.k = (int64_t)o->dptr.size() - 1;
    pub.d_ptr = o->dptr.data();
    pub.d_pos = o->dpos.data();
    pub.c = o->c.data();
    *out = &owned->pub;
    return NET_OK;
}

int32_t net_compressed_free(net_compressed* c) {
    if (c) {
        Owned* owned = reinterpret_cast<Owned*>(c);
        delete owned->st;
        delete owned;
    }
    return NET_OK;
}

}  // extern "C"
#pragma GCC visibility pop
