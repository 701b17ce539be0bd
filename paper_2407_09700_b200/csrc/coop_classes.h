// coop_classes.h -- the l-classes served by the cooperative family (coop_kernel.cuh), split into groups = translation units.
#pragma once
#define COOP_GROUP0(X) X(2,1,1,1) X(2,1,2,0) X(2,1,2,1) X(2,2,2,1)
#define COOP_GROUP1(X) X(3,2,2,1) X(2,2,2,2) X(3,1,2,1) X(3,3,2,1)
